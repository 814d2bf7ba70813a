/* qmc_oracle.h -- CPU oracle for the Slater-Jastrow Psi / E_L / Metropolis path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this library.  It
 * shares no code, header, table or helper with the CUDA path
 * (paper_2506_09743_b200/csrc, include/qmc.h); the struct below is declared
 * here on its own.
 *
 * Everything is float64, long-hand loops, every determinant factored
 * explicitly; no excitation tables, no combined one-body operator, no BLAS.
 * Citations are PAPER.md:<line> (+ equation) of /root/reference/PAPER.md.
 *
 * Parity pins (tests/test_oracle_pins.py): hydrogenic closed forms for every
 * harmonic (1s, 2s, 2p x3, 3d x5), He-like closed form with the Pade Jastrow,
 * n-electron hydrogenic determinants (exact sum of orbital energies), central
 * finite differences of the plain Psi, antisymmetry, Leibniz determinants,
 * nuclear repulsion, cusp finiteness, Philox known answers, sampler moments;
 * parameter derivatives (eq. 6): central differences of log|Psi| in every
 * parameter, sum rule sum_n d_n O_n = 1, He-like closed form, zero gradient for
 * an exact eigenfunction.
 * Unpinned by anything but those: absolute energies of the random-MO
 * synthetic LiH / Li2 / CO configs (no physical reference exists for them).
 */
#ifndef QMC_ORACLE_H
#define QMC_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int32_t n_atoms;
  const double *atom_xyz; /* [n_atoms][3] bohr */
  const double *atom_Z;   /* [n_atoms] */
  int32_t n_up, n_dn;     /* electrons 0..n_up-1 are spin-up */
  int32_t n_ao;
  const int32_t *ao_atom, *ao_n, *ao_l, *ao_m; /* per AO: centre, n, l, harmonic index */
  const double *ao_zeta;  /* [n_ao] */
  const double *ao_norm;  /* [n_ao] or NULL = standard normalisation */
  int32_t n_mo;
  const double *mo_coeff; /* [n_ao][n_mo] */
  int32_t n_det;
  const int32_t *det_up, *det_dn; /* [n_det][n_up], [n_det][n_dn] ordered MO columns */
  const double *ci_coeff;         /* [n_det] */
  double jastrow_a_par, jastrow_a_anti, jastrow_b;
  /* electron-nucleus kernel (D.2): K_en(r) = (w0 r + w1 r^2) / (1 + w2 r), all zero = absent */
  double jastrow_en_w0, jastrow_en_w1, jastrow_en_w2;
  /* electron-electron-nucleus kernel (D.3): n_een terms, each 7 doubles
   * (c, a1, b1, a2, b2, a3, b3):  K_een = sum_mu c [a1 r_ai/(1+b1 r_ai)] [a2 r_aj/(1+b2 r_aj)] [a3 r_ij/(1+b3 r_ij)],
   * summed over every nucleus a and every electron pair once (eq. 5: sum_{alpha, i>j}), each pair
   * symmetrised, 1/2 [K(r_ai, r_aj, r_ij) + K(r_aj, r_ai, r_ij)] (reading Q22: equal to the literal sum when the first
   * two factors coincide, exchange-symmetric when they do not); n_een = 0 = absent */
  int32_t n_een;
  const double *een_params; /* [n_een][7] or NULL */
  /* inverse backflow: rt_i = r_i + sum_{j != i} (w / r_ij)(r_i - r_j) over all other electrons; the
   * orbitals are evaluated at rt, the Jastrow factor at r; 0 = no backflow */
  double backflow_w;
} oracle_system_desc_t;

/* All pointers are HOST pointers.  Walker arrays are SoA [n_e][3][M]; the
 * functions below process walkers w0 <= w < w1 only (so a caller can split a
 * batch over threads) and index every per-walker array with the GLOBAL w. */

/* STO normalisation, reading Q2 (PAPER.md:55 leaves N unspecified). */
double oracle_sto_norm(int n, int l, int m, double zeta);

/* One AO at one point: out = {phi, dphi/dx, dphi/dy, dphi/dz, lap phi}.  PAPER.md:55. */
void oracle_ao_eval(const oracle_system_desc_t *s, int ao, const double *xyz, double *out5);

/* Partial-pivot LU determinant and inverse of a row-major n x n matrix.
 * inv may be NULL.  Returns det. */
double oracle_det_inv(int n, const double *A, double *inv);

/* Plain definition of eq. 4: e^J * sum_n d_n det(A_n^up) det(A_n^dn)
 * for ONE walker given as AoS r[n_e][3].  Used for finite differences. */
double oracle_psi_plain(const oracle_system_desc_t *s, const double *r);

/* log|Psi|, sign, E_L = H Psi / Psi (eq. 1; F.1-F.4, G.7; with backflow_w != 0 the general formulas:
 * F.4 with its cross term and F.5, coordinate by coordinate on every determinant).
 * parts, if non-NULL, receives [M][4] = {kinetic, V_ee, V_en, V_nn}. */
int oracle_local_energy(const oracle_system_desc_t *s, const double *r, int64_t M, int64_t w0,
                        int64_t w1, double *logpsi, double *sign, double *eloc, double *parts);

/* Philox4x32-10 (reading Q9). */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* The proposal normals of walker w at absolute sweep index `sweep`:
 * z[0..n_coord-1] (reading Q9), and the accept uniform. */
void oracle_walker_draws(uint64_t seed, int64_t w, uint64_t sweep, int n_coord, double *z,
                         double *u_accept);

/* All-electron Metropolis (readings Q9, Q10).  r is updated in
 * place.  accept [n_sweeps][M] (uint8) and margin [n_sweeps][M]
 * (= 2*dlog|Psi| - log u, the quantity whose sign is the decision) may be
 * NULL; eloc_acc [M] (sum over sweeps of E_L after each sweep) may be NULL. */
int oracle_metropolis(const oracle_system_desc_t *s, double *r, int64_t M, int64_t w0, int64_t w1,
                      double step, int32_t n_sweeps, uint64_t seed, uint64_t sweep_offset,
                      double *logpsi, double *sign, uint8_t *accept, double *margin,
                      double *eloc_acc);

/* Mean and standard error of the mean (eq. 3), Kahan sums. */
void oracle_batch_stats(const double *x, int64_t M, double *mean, double *stderr_out);

/* Logarithmic derivatives O_p(r) = (d Psi / d theta_p) / Psi, the factor of eq. 6
 * (PAPER.md:78), for theta = (jastrow_a_par, jastrow_a_anti, jastrow_b, jastrow_en_w0, jastrow_en_w1,
 * jastrow_en_w2, then the seven parameters c, a_f, b_f, a_g, b_g, a_h, b_h of every e-e-n term (D.3,
 * PAPER.md:251) in een_params order, then d_0 .. d_{n_det-1}); O is [M][6 + 7 n_een + n_det] row-major,
 * rows w0 <= w < w1 are written.
 * Psi = e^J Sigma (eq. 4), so d ln Psi / d(Jastrow parameter) is the
 * parameter derivative of D.1 summed over pairs, and
 * d ln Psi / d d_n = D_n^up D_n^dn / Sigma, every determinant factored explicitly.
 * With backflow_w != 0 the determinants sit at the backflow coordinates and ONE MORE entry
 * follows the CI entries, the backflow weight: d ln Psi / d w = sum_n d_n D_n [Tr(A_n^-1 d_w A_n)^up + (..)^dn] / Sigma
 * with d_w A[i][j] = grad phi_j(rt_i) . sum_{j' != i} (r_i - r_j') / r_ij'; O is then [M][6 + 7 n_een + n_det + 1]. */
int oracle_log_derivatives(const oracle_system_desc_t *s, const double *r, int64_t M, int64_t w0,
                           int64_t w1, double *O);

/* Logarithmic derivatives with respect to the orbital parameters (eq. 6 factors for the AO and MO layers,
 * PAPER.md:55-57): dC [M][n_ao][n_mo] = d ln Psi / d C[beta][alpha] (the derivative in the scaling mu_{beta,alpha}
 * of PAPER.md:57 is c_{beta,alpha} times it) and dzeta [M][n_ao] = d ln Psi / d zeta_beta, each AO's exponent on
 * its own; the standard normalisation depends on zeta, (2 zeta)^(n+1/2): d ln N / d zeta = (n + 1/2) / zeta, a
 * caller-supplied ao_norm does not.  Every determinant is inverted explicitly:
 *   d ln Sigma / d A_n[i][j] = A_n^-1[j][i]  =>  Gamma[i][alpha] = sum_n w_n A_n^-1[pos_n(alpha)][i],
 *   w_n = d_n D_n^up D_n^dn / Sigma;  dC[beta][alpha] = sum_i ao_beta(r_i) Gamma[i][alpha];
 *   dzeta[beta] = sum_alpha C[beta][alpha] sum_i (d ao_beta / d zeta)(r_i) Gamma[i][alpha].
 * Either output may be NULL.  Rows w0 <= w < w1. 
 * With backflow_w != 0 the orbitals (and their derivatives) are evaluated at the backflow coordinates, which depend on
 * none of these parameters; the Jastrow factor stays at r. */
int oracle_orbital_derivatives(const oracle_system_desc_t *s, const double *r, int64_t M, int64_t w0,
                               int64_t w1, double *dC, double *dzeta);

/* Nuclear log-gradient grad_alpha ln|Psi| = (1/2) grad_alpha ln rho, the factor of the second term of the force
 * estimator (eq. 7), with the atomic positions as parameters of the AO layer:
 * dR [M][n_atoms][3].  d ao_beta(r_i) / d R_a = -grad_r ao_beta(r_i) for the AOs of centre a; chain rule through
 * every determinant inverted explicitly (Gamma as in oracle_orbital_derivatives), plus the nuclear dependence of
 * the Jastrow kernels D.2 and D.3.  Rows w0 <= w < w1. 
 * With backflow_w != 0 the orbitals (and their derivatives) are evaluated at the backflow coordinates, which depend on
 * none of these parameters; the Jastrow factor stays at r. */
int oracle_nuclear_log_gradient(const oracle_system_desc_t *s, const double *r, int64_t M, int64_t w0,
                                int64_t w1, double *dR);

/* The backflow coordinates of ONE walker: r, rt AoS [n_e][3]. */
void oracle_backflow_coords(const oracle_system_desc_t *s, const double *r, double *rt);

/* One AO at one point with its second-level derivatives: out14 = {phi, grad[3], lap, Hessian xx yy zz xy yz zx,
 * grad lap [3]}.  PAPER.md:55; needed because d ao / d R = -grad_r ao. */
void oracle_ao_eval2(const oracle_system_desc_t *s, int ao, const double *xyz, double *out14);

/* grad_alpha E_L, the first term of the force estimator (eq. 7): dE [M][n_atoms][3], rows w0 <= w < w1.
 * Pade e-e Jastrow (D.1) only: returns -2 when the e-n / e-e-n kernels are switched on.  Every determinant is
 * inverted explicitly and the chain rule is applied long-hand to what oracle_local_energy evaluates. */
int oracle_nuclear_energy_gradient(const oracle_system_desc_t *s, const double *r, int64_t M, int64_t w0,
                                   int64_t w1, double *dE);

/* Force estimator of eq. 7 (reading Q23):
 *   F_alpha = -(1/M) sum_m [grad_alpha E_L + 2 (E_L - E_v) grad_alpha ln|Psi|].
 * eloc [M]; dE, dlnpsi [M][n_atoms][3]; F [n_atoms][3]; terms [2][n_atoms][3] (the two contributions) may be NULL. */
void oracle_force(const double *eloc, const double *dE, const double *dlnpsi, int64_t M, int32_t n_atoms,
                  double *F, double *terms);

/* Estimator of eq. 6: E_v = mean E_L, grad_p = (2/M) sum_m O[m][p] (E_L[m] - E_v).
 * Kahan sums.  Ev may be NULL. */
void oracle_energy_gradient(const double *eloc, const double *O, int64_t M, int32_t n_param,
                            double *Ev, double *grad);

#ifdef __cplusplus
}
#endif
#endif
