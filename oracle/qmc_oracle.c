/* qmc_oracle.c -- plain CPU oracle, float64 unless built as the extended-precision adjudicator (see qmc_oracle.h: test
 * infrastructure only; shares nothing with the CUDA path).
 *
 * Build: gcc -O2 -std=c11 -fPIC -shared -o libqmc_oracle.so qmc_oracle.c -lm
 * (no -ffast-math).  Citations: PAPER.md:<line> of /root/reference/PAPER.md.
 */
#include "qmc_oracle.h"

/* Working precision.  The default build computes in float64 (`real` = double: the oracle proper).  The same source
 * compiled with -DORACLE_REAL="long double" (libqmc_oracle_ld.so, x87 80-bit, 64-bit mantissa) is the EXTENDED run
 * that adjudicates walkers on which two float64 evaluations cannot agree to the parity bound (a nearly singular
 * Slater matrix: DESIGN.md section 2, reading Q24).  No algorithm changes with the type: <tgmath.h> selects the
 * libm routine of the operand type.  Inputs and outputs of the API stay double; the random-number stream of the
 * sampler stays float64 in both builds (it is part of the method's definition, reading Q9). */
#ifndef ORACLE_REAL
#define ORACLE_REAL double
#endif
typedef ORACLE_REAL real;

#include <tgmath.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_PI 3.14159265358979323846

/* ------------------------------------------------------------------ */
/* Atomic orbitals: phi = N * S_lm(d) * r^k * exp(-zeta r), */
/* k = n-1-l (reading Q3), S_lm real solid harmonics in the order       */
/* l=0:{1}; l=1:{x,y,z}; l=2:{xy,yz,zx,x^2-y^2,2z^2-x^2-y^2}.           */
/* ------------------------------------------------------------------ */

static real factorial(int n) {
  real f = 1.0;
  for (int i = 2; i <= n; ++i) f *= (real)i;
  return f;
}

static real sto_norm_r(int n, int l, int m, real zeta) {
  /* radial: (2 zeta)^(n+1/2) / sqrt((2n)!) ; angular: real spherical harmonic constant */
  real radial = pow(2.0 * zeta, (real)n + 0.5) / sqrt(factorial(2 * n));
  real ang = 0.0;
  if (l == 0) ang = 1.0 / (2.0 * sqrt(ORACLE_PI));
  else if (l == 1) ang = sqrt(3.0 / (4.0 * ORACLE_PI));
  else if (l == 2) {
    if (m <= 2) ang = 0.5 * sqrt(15.0 / ORACLE_PI);
    else if (m == 3) ang = 0.25 * sqrt(15.0 / ORACLE_PI);
    else ang = 0.25 * sqrt(5.0 / ORACLE_PI);
  }
  return radial * ang;
}

double oracle_sto_norm(int n, int l, int m, double zeta) { return (double)sto_norm_r(n, l, m, (real)zeta); }

/* S, its gradient and its three pure second derivatives, written out. */
static void solid_harmonic(int l, int m, real x, real y, real z, real *S, real g[3],
                           real h[3]) {
  *S = 0.0;
  g[0] = g[1] = g[2] = 0.0;
  h[0] = h[1] = h[2] = 0.0;
  if (l == 0) {
    *S = 1.0;
  } else if (l == 1) {
    if (m == 0) { *S = x; g[0] = 1.0; }
    if (m == 1) { *S = y; g[1] = 1.0; }
    if (m == 2) { *S = z; g[2] = 1.0; }
  } else if (l == 2) {
    if (m == 0) { *S = x * y; g[0] = y; g[1] = x; }
    if (m == 1) { *S = y * z; g[1] = z; g[2] = y; }
    if (m == 2) { *S = z * x; g[0] = z; g[2] = x; }
    if (m == 3) { *S = x * x - y * y; g[0] = 2.0 * x; g[1] = -2.0 * y; h[0] = 2.0; h[1] = -2.0; }
    if (m == 4) {
      *S = 2.0 * z * z - x * x - y * y;
      g[0] = -2.0 * x; g[1] = -2.0 * y; g[2] = 4.0 * z;
      h[0] = -2.0; h[1] = -2.0; h[2] = 4.0;
    }
  }
}

static void ao_eval_r(const oracle_system_desc_t *s, int ao, const real *xyz, real *out5) {
  int a = s->ao_atom[ao], n = s->ao_n[ao], l = s->ao_l[ao], m = s->ao_m[ao];
  real zeta = s->ao_zeta[ao];
  real N = s->ao_norm ? s->ao_norm[ao] : sto_norm_r(n, l, m, zeta);
  real d[3];
  for (int c = 0; c < 3; ++c) d[c] = xyz[c] - s->atom_xyz[3 * a + c];
  real r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
  int k = n - 1 - l;

  real S, gS[3], hS[3];
  solid_harmonic(l, m, d[0], d[1], d[2], &S, gS, hS);

  /* radial factor f(r) = r^k e^{-zeta r} and its first two derivatives, term by term */
  real e = exp(-zeta * r);
  real rk = pow(r, (real)k);                         /* r^k       */
  real rk1 = (k >= 1) ? pow(r, (real)(k - 1)) : 0.0; /* r^(k-1)   */
  real rk2 = (k >= 2) ? pow(r, (real)(k - 2)) : 0.0; /* r^(k-2)   */
  real f = rk * e;
  real f1 = ((real)k * rk1 - zeta * rk) * e;
  real f2 = ((real)(k * (k - 1)) * rk2 - 2.0 * (real)k * zeta * rk1 + zeta * zeta * rk) * e;

  /* grad f = f' d/r ; lap f = f'' + 2 f'/r */
  real gf[3];
  for (int c = 0; c < 3; ++c) gf[c] = f1 * d[c] / r;
  real lapf = f2 + 2.0 * f1 / r;

  /* product rule: grad(S f) = gS f + S gf ; lap(S f) = lapS f + 2 gS.gf + S lapf */
  real lapS = hS[0] + hS[1] + hS[2];
  real dot = gS[0] * gf[0] + gS[1] * gf[1] + gS[2] * gf[2];
  out5[0] = N * S * f;
  for (int c = 0; c < 3; ++c) out5[1 + c] = N * (gS[c] * f + S * gf[c]);
  out5[4] = N * (lapS * f + 2.0 * dot + S * lapf);
}

void oracle_ao_eval(const oracle_system_desc_t *s, int ao, const double *xyz, double *out5) {
  real p[3] = {xyz[0], xyz[1], xyz[2]}, o[5];
  ao_eval_r(s, ao, p, o);
  for (int q = 0; q < 5; ++q) out5[q] = (double)o[q];
}

/* ------------------------------------------------------------------ */
/* Partial-pivot LU: determinant and inverse   */
/* ------------------------------------------------------------------ */

static real det_inv_r(int n, const real *A, real *inv) {
  if (n <= 0) return 1.0;
  real *lu = (real *)malloc(sizeof(real) * (size_t)n * (size_t)n);
  int *perm = (int *)malloc(sizeof(int) * (size_t)n);
  memcpy(lu, A, sizeof(real) * (size_t)n * (size_t)n);
  for (int i = 0; i < n; ++i) perm[i] = i;
  real det = 1.0;
  for (int k = 0; k < n; ++k) {
    int p = k;
    real best = fabs(lu[k * n + k]);
    for (int i = k + 1; i < n; ++i)
      if (fabs(lu[i * n + k]) > best) { best = fabs(lu[i * n + k]); p = i; }
    if (p != k) {
      for (int j = 0; j < n; ++j) { real t = lu[k * n + j]; lu[k * n + j] = lu[p * n + j]; lu[p * n + j] = t; }
      int t = perm[k]; perm[k] = perm[p]; perm[p] = t;
      det = -det;
    }
    real piv = lu[k * n + k];
    det *= piv;
    if (piv == 0.0) continue; /* singular: det = 0, inverse undefined (inf/nan follow) */
    for (int i = k + 1; i < n; ++i) {
      lu[i * n + k] /= piv;
      real lik = lu[i * n + k];
      for (int j = k + 1; j < n; ++j) lu[i * n + j] -= lik * lu[k * n + j];
    }
  }
  if (inv) {
    /* solve A x = e_c for every unit vector: P A = L U */
    real *y = (real *)malloc(sizeof(real) * (size_t)n);
    for (int c = 0; c < n; ++c) {
      for (int i = 0; i < n; ++i) {
        real v = (perm[i] == c) ? 1.0 : 0.0;
        for (int j = 0; j < i; ++j) v -= lu[i * n + j] * y[j];
        y[i] = v;
      }
      for (int i = n - 1; i >= 0; --i) {
        real v = y[i];
        for (int j = i + 1; j < n; ++j) v -= lu[i * n + j] * inv[j * n + c];
        inv[i * n + c] = v / lu[i * n + i];
      }
    }
    free(y);
  }
  free(lu);
  free(perm);
  return det;
}

double oracle_det_inv(int n, const double *A, double *inv) {
  if (n <= 0) return 1.0;
  size_t nn = (size_t)n * (size_t)n;
  real *a = (real *)malloc(sizeof(real) * nn), *ai = inv ? (real *)malloc(sizeof(real) * nn) : NULL;
  for (size_t i = 0; i < nn; ++i) a[i] = A[i];
  real det = det_inv_r(n, a, ai);
  if (inv)
    for (size_t i = 0; i < nn; ++i) inv[i] = (double)ai[i];
  free(a);
  free(ai);
  return (double)det;
}

/* ------------------------------------------------------------------ */
/* Pade e-e Jastrow (D.1; cusps C.1):       */
/* K(r) = w0 r / (1 + w r), w0 = a_par (same spin), a_anti (opposite).  */
/* ------------------------------------------------------------------ */

static int spin_of(const oracle_system_desc_t *s, int i) { return i < s->n_up ? 0 : 1; }
static void jastrow_een_add(const oracle_system_desc_t *s, const real *r, real *J, real *gJ, real *lapJ);

/* J, grad_i J [n_e][3], lap J (sum over all electrons), pair loop. r is AoS [n_e][3]. */
static void jastrow_all(const oracle_system_desc_t *s, const real *r, real *J, real *gJ,
                        real *lapJ) {
  int ne = s->n_up + s->n_dn;
  *J = 0.0;
  *lapJ = 0.0;
  for (int i = 0; i < 3 * ne; ++i) gJ[i] = 0.0;
  for (int i = 0; i < ne; ++i)
    for (int j = i + 1; j < ne; ++j) {
      real a = (spin_of(s, i) == spin_of(s, j)) ? s->jastrow_a_par : s->jastrow_a_anti;
      real b = s->jastrow_b;
      real d[3];
      for (int c = 0; c < 3; ++c) d[c] = r[3 * i + c] - r[3 * j + c];
      real rij = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
      real den = 1.0 + b * rij;
      real u = a * rij / den;
      real u1 = a / (den * den);
      real u2 = -2.0 * a * b / (den * den * den);
      *J += u;
      for (int c = 0; c < 3; ++c) {
        gJ[3 * i + c] += u1 * d[c] / rij;
        gJ[3 * j + c] -= u1 * d[c] / rij;
      }
      /* lap_i K + lap_j K = 2 (u'' + 2 u'/r) */
      *lapJ += 2.0 * (u2 + 2.0 * u1 / rij);
    }
  /* electron-nucleus kernel (D.2): K_en(r) = N / D, N = w0 r + w1 r^2, D = 1 + w2 r,
   * summed over every (electron, nucleus) pair; quotient rule long-hand */
  real w0 = s->jastrow_en_w0, w1 = s->jastrow_en_w1, w2 = s->jastrow_en_w2;
  if (w0 != 0.0 || w1 != 0.0)
    for (int i = 0; i < ne; ++i)
      for (int at = 0; at < s->n_atoms; ++at) {
        real d[3];
        for (int c = 0; c < 3; ++c) d[c] = r[3 * i + c] - s->atom_xyz[3 * at + c];
        real ria = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        real N = w0 * ria + w1 * ria * ria, D = 1.0 + w2 * ria;
        real N1 = w0 + 2.0 * w1 * ria, N2 = 2.0 * w1, D1 = w2;
        real K = N / D;
        real K1 = (N1 * D - N * D1) / (D * D);
        /* (N'D - N D')' = N''D - N D'' = N''D ;  K'' = N''D / D^2 - 2 D' (N'D - N D') / D^3 */
        real K2 = N2 * D / (D * D) - 2.0 * D1 * (N1 * D - N * D1) / (D * D * D);
        *J += K;
        for (int c = 0; c < 3; ++c) gJ[3 * i + c] += K1 * d[c] / ria;
        *lapJ += K2 + 2.0 * K1 / ria;
      }
  if (s->n_een > 0) jastrow_een_add(s, r, J, gJ, lapJ);
}

/* electron-electron-nucleus kernel (D.3).  Eq. 5 sums K_een over every nucleus and every
 * pair once, sum_{alpha, i>j}.  With different first and second Pade factors the literal K_een(r_ai, r_aj, r_ij) is not
 * symmetric in (i, j), which would break the exchange symmetry of PAPER.md:51, so each pair enters symmetrised
 * (reading Q22):  K_pair = 1/2 [K_een(r_ai, r_aj, r_ij) + K_een(r_aj, r_ai, r_ij)]  -- identical to the paper's literal
 * sum when the two factors coincide.  Written as a loop over ORDERED pairs i != j with weight 1/2.
 * One term T = (c/2) f(r_ai) g(r_aj) h(r_ij), Pade factors p(r) = a r/(1 + b r), p' = a/(1 + b r)^2,
 * p'' = -2 a b/(1 + b r)^3.  Product rule long-hand:
 *   grad_i T = c g [f' h e_ai + f h' e_ij]            e_ai = (r_i - R_a)/r_ai, e_ij = (r_i - r_j)/r_ij
 *   grad_j T = c f [g' h e_aj - g h' e_ij]
 *   lap_i T  = c g [(f'' + 2 f'/r_ai) h + f (h'' + 2 h'/r_ij) + 2 f' h' e_ai.e_ij]
 *   lap_j T  = c f [(g'' + 2 g'/r_aj) h + g (h'' + 2 h'/r_ij) - 2 g' h' e_aj.e_ij]
 * Adds to J, gJ, lapJ; any of gJ / lapJ may be NULL (value only). */
static void pade3(real a, real b, real r, real *p, real *p1, real *p2) {
  real D = 1.0 + b * r;
  *p = a * r / D;
  *p1 = a / (D * D);
  *p2 = -2.0 * a * b / (D * D * D);
}

static void jastrow_een_add(const oracle_system_desc_t *s, const real *r, real *J, real *gJ, real *lapJ) {
  int ne = s->n_up + s->n_dn;
  for (int at = 0; at < s->n_atoms; ++at)
    for (int i = 0; i < ne; ++i)
      for (int j = 0; j < ne; ++j) {
        if (i == j) continue;
        real eai[3], eaj[3], eij[3];
        for (int c = 0; c < 3; ++c) {
          eai[c] = r[3 * i + c] - s->atom_xyz[3 * at + c];
          eaj[c] = r[3 * j + c] - s->atom_xyz[3 * at + c];
          eij[c] = r[3 * i + c] - r[3 * j + c];
        }
        real rai = sqrt(eai[0] * eai[0] + eai[1] * eai[1] + eai[2] * eai[2]);
        real raj = sqrt(eaj[0] * eaj[0] + eaj[1] * eaj[1] + eaj[2] * eaj[2]);
        real rij = sqrt(eij[0] * eij[0] + eij[1] * eij[1] + eij[2] * eij[2]);
        for (int c = 0; c < 3; ++c) { eai[c] /= rai; eaj[c] /= raj; eij[c] /= rij; }
        real ai_ij = eai[0] * eij[0] + eai[1] * eij[1] + eai[2] * eij[2];
        real aj_ij = eaj[0] * eij[0] + eaj[1] * eij[1] + eaj[2] * eij[2];
        for (int mu = 0; mu < s->n_een; ++mu) {
          const double *q = s->een_params + 7 * mu;
          real f, f1, f2, g, g1, g2, h, h1, h2;
          pade3(q[1], q[2], rai, &f, &f1, &f2);
          pade3(q[3], q[4], raj, &g, &g1, &g2);
          pade3(q[5], q[6], rij, &h, &h1, &h2);
          real ch = 0.5 * q[0]; /* each unordered pair is visited twice, as (i,j) and as (j,i) */
          *J += ch * f * g * h;
          if (gJ)
            for (int c = 0; c < 3; ++c) {
              gJ[3 * i + c] += ch * g * (f1 * h * eai[c] + f * h1 * eij[c]);
              gJ[3 * j + c] += ch * f * (g1 * h * eaj[c] - g * h1 * eij[c]);
            }
          if (lapJ) {
            *lapJ += ch * g * ((f2 + 2.0 * f1 / rai) * h + f * (h2 + 2.0 * h1 / rij) + 2.0 * f1 * h1 * ai_ij);
            *lapJ += ch * f * ((g2 + 2.0 * g1 / raj) * h + g * (h2 + 2.0 * h1 / rij) - 2.0 * g1 * h1 * aj_ij);
          }
        }
      }
}

/* value of the electron-nucleus part of J alone (D.2) */
static real jastrow_en_value(const oracle_system_desc_t *s, const real *r) {
  int ne = s->n_up + s->n_dn;
  real J = 0.0;
  for (int i = 0; i < ne; ++i)
    for (int at = 0; at < s->n_atoms; ++at) {
      real dx = r[3 * i] - s->atom_xyz[3 * at], dy = r[3 * i + 1] - s->atom_xyz[3 * at + 1],
             dz = r[3 * i + 2] - s->atom_xyz[3 * at + 2];
      real ria = sqrt(dx * dx + dy * dy + dz * dz);
      J += (s->jastrow_en_w0 * ria + s->jastrow_en_w1 * ria * ria) / (1.0 + s->jastrow_en_w2 * ria);
    }
  return J;
}

/* ------------------------------------------------------------------ */
/* Backflow transformation:                               */
/*   rt_i = r_i + sum_{j != i} K_BF(r_ij) (r_i - r_j),  over ALL other   */
/* electrons, with the inverse kernel K_BF(r) = w / r.     */
/* The orbitals are evaluated at rt, the Jastrow factor at r (PAPER.md:  */
/* 61).  With t_a(d) = K(|d|) d_a, d = r_i - r_j:                         */
/*   d_b t_a     = K' d_a d_b / r + K delta_ab                            */
/*   d_b d_b t_a = K'' d_b^2 d_a / r^2 + K' d_a (1/r - d_b^2/r^3)         */
/*                 + 2 K' d_b delta_ab / r                                */
/* and d/dx_i = +d/dd, d/dx_j = -d/dd.  Outputs (any may be NULL):       */
/*   rt  [ne][3];  jac [ne][3][3 ne] = d rt_i^a / d x_l  (l = 3 m + b);   */
/*   lap2 [ne][3][3 ne] = d^2 rt_i^a / d x_l^2.                           */
/* ------------------------------------------------------------------ */
static void backflow_kernel(real w, real r, real *K, real *K1, real *K2) {
  *K = w / r;
  *K1 = -w / (r * r);
  *K2 = 2.0 * w / (r * r * r);
}

static void backflow_map(const oracle_system_desc_t *s, const real *r, real *rt, real *jac, real *lap2) {
  int ne = s->n_up + s->n_dn, nc = 3 * ne;
  real w = s->backflow_w;
  if (jac)
    for (int q = 0; q < ne * 3 * nc; ++q) jac[q] = 0.0;
  if (lap2)
    for (int q = 0; q < ne * 3 * nc; ++q) lap2[q] = 0.0;
  for (int i = 0; i < ne; ++i) {
    for (int a = 0; a < 3; ++a) {
      rt[3 * i + a] = r[3 * i + a];
      if (jac) jac[(3 * i + a) * nc + 3 * i + a] = 1.0;
    }
    for (int j = 0; j < ne; ++j) {
      if (j == i) continue;
      real d[3];
      for (int a = 0; a < 3; ++a) d[a] = r[3 * i + a] - r[3 * j + a];
      real rij = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
      real K, K1, K2;
      backflow_kernel(w, rij, &K, &K1, &K2);
      for (int a = 0; a < 3; ++a) {
        rt[3 * i + a] += K * d[a];
        for (int b = 0; b < 3; ++b) {
          real dl = (a == b) ? 1.0 : 0.0;
          real t1 = K1 * d[a] * d[b] / rij + K * dl;
          real t2 = K2 * d[b] * d[b] * d[a] / (rij * rij) + K1 * d[a] * (1.0 / rij - d[b] * d[b] / (rij * rij * rij)) +
                    2.0 * K1 * d[b] * dl / rij;
          if (jac) {
            jac[(3 * i + a) * nc + 3 * i + b] += t1;
            jac[(3 * i + a) * nc + 3 * j + b] -= t1;
          }
          if (lap2) {
            lap2[(3 * i + a) * nc + 3 * i + b] += t2;
            lap2[(3 * i + a) * nc + 3 * j + b] += t2;
          }
        }
      }
    }
  }
}

void oracle_backflow_coords(const oracle_system_desc_t *s, const double *r_in, double *rt_out) {
  int ne = s->n_up + s->n_dn;
  real *r = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1)), *rt = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  for (int q = 0; q < 3 * ne; ++q) r[q] = r_in[q];
  backflow_map(s, r, rt, NULL, NULL);
  for (int q = 0; q < 3 * ne; ++q) rt_out[q] = (double)rt[q];
  free(r); free(rt);
}

static void ao_eval2_r(const oracle_system_desc_t *s, int ao, const real *xyz, real *out14);
static void local_energy_backflow_one(const oracle_system_desc_t *s, const real *r, real *logpsi, real *sign, real *eloc,
                                      real *parts);

/* ------------------------------------------------------------------ */
/* AO -> MO: phi_alpha = sum_beta C[beta][alpha] ao_beta  */
/* mo[i][alpha][q], q = value, d/dx, d/dy, d/dz, laplacian              */
/* ------------------------------------------------------------------ */

static void mo_all(const oracle_system_desc_t *s, const real *r, real *mo) {
  int ne = s->n_up + s->n_dn;
  real ao[5];
  for (int i = 0; i < ne * s->n_mo * 5; ++i) mo[i] = 0.0;
  for (int i = 0; i < ne; ++i)
    for (int beta = 0; beta < s->n_ao; ++beta) {
      ao_eval_r(s, beta, r + 3 * i, ao);
      for (int alpha = 0; alpha < s->n_mo; ++alpha)
        for (int q = 0; q < 5; ++q)
          mo[(i * s->n_mo + alpha) * 5 + q] += s->mo_coeff[beta * s->n_mo + alpha] * ao[q];
    }
}

double oracle_psi_plain(const oracle_system_desc_t *s, const double *r_in) {
  int ne = s->n_up + s->n_dn, nmo = s->n_mo;
  real *r = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  for (int i = 0; i < 3 * ne; ++i) r[i] = r_in[i];
  real *mo = (real *)malloc(sizeof(real) * (size_t)(ne * nmo * 5 + 1));
  real *gJ = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  real *A = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  if (s->backflow_w != 0.0) { /* orbitals at the backflow coordinates, Jastrow at the electrons' own */
    real *rt = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
    backflow_map(s, r, rt, NULL, NULL);
    mo_all(s, rt, mo);
    free(rt);
  } else {
    mo_all(s, r, mo);
  }
  real J, lapJ;
  jastrow_all(s, r, &J, gJ, &lapJ);
  real sigma = 0.0;
  for (int n = 0; n < s->n_det; ++n) {
    real D[2];
    for (int sp = 0; sp < 2; ++sp) {
      int ns = sp ? s->n_dn : s->n_up, e0 = sp ? s->n_up : 0;
      const int32_t *lst = sp ? s->det_dn + (size_t)n * s->n_dn : s->det_up + (size_t)n * s->n_up;
      for (int i = 0; i < ns; ++i)
        for (int j = 0; j < ns; ++j) A[i * ns + j] = mo[((e0 + i) * nmo + lst[j]) * 5 + 0];
      D[sp] = det_inv_r(ns, A, NULL);
    }
    sigma += s->ci_coeff[n] * D[0] * D[1];
  }
  free(mo); free(gJ); free(A); free(r);
  return (double)(exp(J) * sigma);
}

/* ------------------------------------------------------------------ */
/* Local energy of one walker (AoS r[n_e][3]).                          */
/* F.1, F.2 (:295), F.3 (:300), F.4 (:304), G.7 (:386),  */
/* eq. 1 (:21).                                                         */
/* ------------------------------------------------------------------ */

static void local_energy_one(const oracle_system_desc_t *s, const real *r, real *work,
                             real *logpsi, real *sign, real *eloc, real *parts) {
  int ne = s->n_up + s->n_dn, nmo = s->n_mo;
  real *mo = work;                 /* ne*nmo*5 */
  real *gJ = mo + ne * nmo * 5;    /* 3 ne */
  real *gS = gJ + 3 * ne;          /* 3 ne: grad_i Sigma */
  real *A = gS + 3 * ne;           /* ne*ne */
  real *Ai = A + ne * ne;          /* ne*ne */
  real *gdet = Ai + ne * ne;       /* 3 ne: grad_i D / D of the current determinant */

  if (s->backflow_w != 0.0) { /* every row of A depends on every electron: the general formulas (F.4 cross term, F.5) */
    local_energy_backflow_one(s, r, logpsi, sign, eloc, parts);
    return;
  }
  mo_all(s, r, mo);
  real J, lapJ;
  jastrow_all(s, r, &J, gJ, &lapJ);

  real sigma = 0.0, lapS = 0.0;
  for (int i = 0; i < 3 * ne; ++i) gS[i] = 0.0;
  for (int n = 0; n < s->n_det; ++n) {
    real D[2], t[2];
    for (int sp = 0; sp < 2; ++sp) {
      int ns = sp ? s->n_dn : s->n_up, e0 = sp ? s->n_up : 0;
      const int32_t *lst = sp ? s->det_dn + (size_t)n * s->n_dn : s->det_up + (size_t)n * s->n_up;
      /* rows = electrons, columns = orbitals (reading Q7) */
      for (int i = 0; i < ns; ++i)
        for (int j = 0; j < ns; ++j) A[i * ns + j] = mo[((e0 + i) * nmo + lst[j]) * 5 + 0];
      D[sp] = det_inv_r(ns, A, Ai);
      t[sp] = 0.0;
      for (int i = 0; i < ns; ++i) {
        /* G.2: Tr(A^-1 dA/dx_i) = sum_k A^-1[k][i] d phi_k(r_i)/dx_i ; G.7 likewise with lap */
        for (int c = 0; c < 3; ++c) {
          real g = 0.0;
          for (int k = 0; k < ns; ++k) g += Ai[k * ns + i] * mo[((e0 + i) * nmo + lst[k]) * 5 + 1 + c];
          gdet[3 * (e0 + i) + c] = g;
        }
        for (int k = 0; k < ns; ++k) t[sp] += Ai[k * ns + i] * mo[((e0 + i) * nmo + lst[k]) * 5 + 4];
      }
    }
    real w = s->ci_coeff[n] * D[0] * D[1];
    sigma += w;
    for (int i = 0; i < 3 * ne; ++i) gS[i] += w * gdet[i];   /* F.2 */
    lapS += w * (t[0] + t[1]);                               /* F.4; cross term vanishes (no coordinate in both spins) */
  }

  /* F.1 with script-J = e^J (reading Q5): lap Psi / Psi = lapJ + |gJ|^2 + 2 gJ.gS/S + lapS/S */
  real gJ2 = 0.0, cross = 0.0;
  for (int i = 0; i < 3 * ne; ++i) { gJ2 += gJ[i] * gJ[i]; cross += gJ[i] * gS[i]; }
  real lap_over_psi = lapJ + gJ2 + 2.0 * cross / sigma + lapS / sigma;
  real kinetic = -0.5 * lap_over_psi;

  /* potential, eq. 1 */
  real vee = 0.0, ven = 0.0, vnn = 0.0;
  for (int i = 0; i < ne; ++i)
    for (int j = i + 1; j < ne; ++j) {
      real dx = r[3 * i] - r[3 * j], dy = r[3 * i + 1] - r[3 * j + 1], dz = r[3 * i + 2] - r[3 * j + 2];
      vee += 1.0 / sqrt(dx * dx + dy * dy + dz * dz);
    }
  for (int i = 0; i < ne; ++i)
    for (int a = 0; a < s->n_atoms; ++a) {
      real dx = r[3 * i] - s->atom_xyz[3 * a], dy = r[3 * i + 1] - s->atom_xyz[3 * a + 1],
             dz = r[3 * i + 2] - s->atom_xyz[3 * a + 2];
      ven -= s->atom_Z[a] / sqrt(dx * dx + dy * dy + dz * dz);
    }
  for (int a = 0; a < s->n_atoms; ++a)
    for (int b = a + 1; b < s->n_atoms; ++b) {
      real dx = s->atom_xyz[3 * a] - s->atom_xyz[3 * b], dy = s->atom_xyz[3 * a + 1] - s->atom_xyz[3 * b + 1],
             dz = s->atom_xyz[3 * a + 2] - s->atom_xyz[3 * b + 2];
      vnn += s->atom_Z[a] * s->atom_Z[b] / sqrt(dx * dx + dy * dy + dz * dz);
    }

  *logpsi = J + log(fabs(sigma));
  *sign = (sigma > 0.0) ? 1.0 : ((sigma < 0.0) ? -1.0 : 0.0);
  *eloc = kinetic + vee + ven + vnn;
  if (parts) { parts[0] = kinetic; parts[1] = vee; parts[2] = ven; parts[3] = vnn; }
}

static size_t work_doubles(const oracle_system_desc_t *s) {
  size_t ne = (size_t)(s->n_up + s->n_dn);
  return ne * (size_t)s->n_mo * 5 + 9 * ne + 2 * ne * ne + 16;
}

static void gather_walker(const double *r, int64_t M, int64_t w, int ne, real *aos) {
  for (int i = 0; i < ne; ++i)
    for (int c = 0; c < 3; ++c) aos[3 * i + c] = r[((size_t)i * 3 + (size_t)c) * (size_t)M + (size_t)w];
}

int oracle_local_energy(const oracle_system_desc_t *s, const double *r, int64_t M, int64_t w0,
                        int64_t w1, double *logpsi, double *sign, double *eloc, double *parts) {
  int ne = s->n_up + s->n_dn;
  real *work = (real *)malloc(sizeof(real) * work_doubles(s));
  real *pos = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  if (!work || !pos) return -1;
  for (int64_t w = w0; w < w1; ++w) {
    gather_walker(r, M, w, ne, pos);
    real lp, sg, el, p4[4];
    local_energy_one(s, pos, work, &lp, &sg, &el, parts ? p4 : NULL);
    if (parts)
      for (int q = 0; q < 4; ++q) parts[4 * w + q] = (double)p4[q];
    if (logpsi) logpsi[w] = (double)lp;
    if (sign) sign[w] = (double)sg;
    if (eloc) eloc[w] = (double)el;
  }
  free(work); free(pos);
  return 0;
}

/* ------------------------------------------------------------------ */
/* Philox4x32-10 counter-based generator (reading Q9)                   */
/* ------------------------------------------------------------------ */

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* two words -> u in (0,1): ((hi*2^32 + lo) >> 11 + 1/2) * 2^-53 */
static double uniform53(uint32_t hi, uint32_t lo) {
  uint64_t v = (((uint64_t)hi << 32) | (uint64_t)lo) >> 11;
  return ((double)v + 0.5) * (1.0 / 9007199254740992.0);
}

void oracle_walker_draws(uint64_t seed, int64_t w, uint64_t sweep, int n_coord, double *z,
                         double *u_accept) {
  uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
  uint32_t ctr[4], out[4];
  ctr[0] = (uint32_t)((uint64_t)w & 0xFFFFFFFFu);
  ctr[1] = (uint32_t)(sweep & 0xFFFFFFFFu);
  ctr[3] = (uint32_t)((uint64_t)w >> 32);
  int n_pairs = (n_coord + 1) / 2;
  for (int j = 0; j < n_pairs; ++j) {
    ctr[2] = (uint32_t)j;
    oracle_philox4x32_10(ctr, key, out);
    double u1 = uniform53(out[0], out[1]);
    double u2 = uniform53(out[2], out[3]);
    /* Box-Muller */
    double rho = sqrt(-2.0 * log(u1));
    double theta = 2.0 * ORACLE_PI * u2;
    if (z) {
      z[2 * j] = rho * cos(theta);
      if (2 * j + 1 < n_coord) z[2 * j + 1] = rho * sin(theta);
    }
  }
  if (u_accept) {
    ctr[2] = 0xFFFFFFFFu;
    oracle_philox4x32_10(ctr, key, out);
    *u_accept = uniform53(out[0], out[1]);
  }
}

/* ------------------------------------------------------------------ */
/* log|Psi| and sign from the plain definition (eq. 4)     */
/* ------------------------------------------------------------------ */

static void logpsi_one(const oracle_system_desc_t *s, const real *r, real *work, real *logpsi,
                       real *sign) {
  int ne = s->n_up + s->n_dn, nmo = s->n_mo;
  real *mo = work;              /* ne*nmo (values only) */
  real *A = mo + ne * nmo * 5;  /* ne*ne, same offsets as local_energy_one's layout */
  real ao[5];
  real *rt = A + ne * ne;        /* 3 ne: orbital arguments (the backflow coordinates, or r itself) */
  if (s->backflow_w != 0.0) backflow_map(s, r, rt, NULL, NULL);
  else
    for (int q = 0; q < 3 * ne; ++q) rt[q] = r[q];
  for (int i = 0; i < ne * nmo; ++i) mo[i] = 0.0;
  for (int i = 0; i < ne; ++i)
    for (int beta = 0; beta < s->n_ao; ++beta) {
      ao_eval_r(s, beta, rt + 3 * i, ao);
      for (int alpha = 0; alpha < nmo; ++alpha) mo[i * nmo + alpha] += s->mo_coeff[beta * nmo + alpha] * ao[0];
    }
  real J = 0.0;
  for (int i = 0; i < ne; ++i)
    for (int j = i + 1; j < ne; ++j) {
      real a = (spin_of(s, i) == spin_of(s, j)) ? s->jastrow_a_par : s->jastrow_a_anti;
      real dx = r[3 * i] - r[3 * j], dy = r[3 * i + 1] - r[3 * j + 1], dz = r[3 * i + 2] - r[3 * j + 2];
      real rij = sqrt(dx * dx + dy * dy + dz * dz);
      J += a * rij / (1.0 + s->jastrow_b * rij);
    }
  J += jastrow_en_value(s, r);
  if (s->n_een > 0) jastrow_een_add(s, r, &J, NULL, NULL);
  real sigma = 0.0;
  for (int n = 0; n < s->n_det; ++n) {
    real D[2];
    for (int sp = 0; sp < 2; ++sp) {
      int ns = sp ? s->n_dn : s->n_up, e0 = sp ? s->n_up : 0;
      const int32_t *lst = sp ? s->det_dn + (size_t)n * s->n_dn : s->det_up + (size_t)n * s->n_up;
      for (int i = 0; i < ns; ++i)
        for (int j = 0; j < ns; ++j) A[i * ns + j] = mo[(e0 + i) * nmo + lst[j]];
      D[sp] = det_inv_r(ns, A, NULL);
    }
    sigma += s->ci_coeff[n] * D[0] * D[1];
  }
  *logpsi = J + log(fabs(sigma));
  *sign = (sigma > 0.0) ? 1.0 : ((sigma < 0.0) ? -1.0 : 0.0);
}

/* ------------------------------------------------------------------ */
/* All-electron Metropolis (readings Q9, Q10)             */
/* ------------------------------------------------------------------ */

int oracle_metropolis(const oracle_system_desc_t *s, double *r, int64_t M, int64_t w0, int64_t w1,
                      double step, int32_t n_sweeps, uint64_t seed, uint64_t sweep_offset,
                      double *logpsi, double *sign, uint8_t *accept, double *margin,
                      double *eloc_acc) {
  int ne = s->n_up + s->n_dn, nc = 3 * ne;
  real *work = (real *)malloc(sizeof(real) * work_doubles(s));
  real *pos = (real *)malloc(sizeof(real) * (size_t)(nc + 1));
  real *prop = (real *)malloc(sizeof(real) * (size_t)(nc + 1));
  double *z = (double *)malloc(sizeof(double) * (size_t)(nc + 2));
  if (!work || !pos || !prop || !z) return -1;
  for (int64_t w = w0; w < w1; ++w) {
    gather_walker(r, M, w, ne, pos);
    real lp, sg;
    logpsi_one(s, pos, work, &lp, &sg);
    real acc_e = 0.0;
    for (int32_t sw = 0; sw < n_sweeps; ++sw) {
      double u;
      oracle_walker_draws(seed, w, sweep_offset + (uint64_t)sw, nc, z, &u);
      /* the walker's state is float64 in every build: the move is rounded to double */
      for (int q = 0; q < nc; ++q) prop[q] = (real)((double)pos[q] + step * z[q]);
      real lp2, sg2;
      logpsi_one(s, prop, work, &lp2, &sg2);
      real mg = 2.0 * (lp2 - lp) - log(u);
      int ok = (log(u) < 2.0 * (lp2 - lp)) ? 1 : 0; /* false for NaN and for Psi' = 0 */
      if (ok) {
        for (int q = 0; q < nc; ++q) pos[q] = prop[q];
        lp = lp2;
        sg = sg2;
      }
      if (accept) accept[(size_t)sw * (size_t)M + (size_t)w] = (uint8_t)ok;
      if (margin) margin[(size_t)sw * (size_t)M + (size_t)w] = (double)mg;
      if (eloc_acc) {
        real l3, s3, el;
        local_energy_one(s, pos, work, &l3, &s3, &el, NULL);
        acc_e += el;
      }
    }
    for (int i = 0; i < ne; ++i)
      for (int c = 0; c < 3; ++c) r[((size_t)i * 3 + (size_t)c) * (size_t)M + (size_t)w] = (double)pos[3 * i + c];
    if (logpsi) logpsi[w] = (double)lp;
    if (sign) sign[w] = (double)sg;
    if (eloc_acc) eloc_acc[w] = (double)acc_e;
  }
  free(work); free(pos); free(prop); free(z);
  return 0;
}

/* ------------------------------------------------------------------ */
/* Batch statistics (eq. 3), Kahan-compensated             */
/* ------------------------------------------------------------------ */

void oracle_batch_stats(const double *x, int64_t M, double *mean, double *stderr_out) {
  double sum = 0.0, comp = 0.0;
  for (int64_t i = 0; i < M; ++i) {
    double y = x[i] - comp, t = sum + y;
    comp = (t - sum) - y;
    sum = t;
  }
  double mu = sum / (double)M;
  double s2 = 0.0;
  comp = 0.0;
  for (int64_t i = 0; i < M; ++i) {
    double dlt = x[i] - mu;
    double y = dlt * dlt - comp, t = s2 + y;
    comp = (t - s2) - y;
    s2 = t;
  }
  if (mean) *mean = mu;
  if (stderr_out) *stderr_out = (M > 1) ? sqrt(s2 / (double)(M - 1) / (double)M) : 0.0;
}

/* ------------------------------------------------------------------ */
/* Parameter derivatives of ln Psi and the gradient estimator (eq. 6,   */
/* PAPER.md:78).  theta = (a_par, a_anti, b, en_w0, en_w1, en_w2, d_n). */
/* ------------------------------------------------------------------ */

int oracle_log_derivatives(const oracle_system_desc_t *s, const double *r, int64_t M, int64_t w0,
                           int64_t w1, double *O) {
  /* With the backflow transformation the Jastrow entries are unchanged (the Jastrow factor sits at r),
   * the orbitals of the CI entries sit at the backflow coordinates, and one more entry follows them: the backflow
   * weight w of K_BF(r) = w / r,
   *   d ln Psi / d w = sum_n d_n D_n^up D_n^dn [Tr(A_n^-1 d_w A_n)^up + (..)^dn] / Sigma,
   *   d_w A[i][j] = grad phi_j(rt_i) . d rt_i / d w,   d rt_i / d w = sum_{j != i} (r_i - r_j) / r_ij. */
  const int bf = s->backflow_w != 0.0;
  int ne = s->n_up + s->n_dn, nmo = s->n_mo, nj = 6 + 7 * s->n_een, np = nj + s->n_det + (bf ? 1 : 0);
  real *mo = (real *)malloc(sizeof(real) * (size_t)(ne * nmo + 1));
  real *dmo = (real *)malloc(sizeof(real) * (size_t)(ne * nmo + 1));
  real *A = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *Ai = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *pos = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  real *post = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  real *prod = (real *)malloc(sizeof(real) * (size_t)(s->n_det + 1));
  if (!mo || !dmo || !A || !Ai || !pos || !post || !prod) return -1;
  real ao[5];
  for (int64_t w = w0; w < w1; ++w) {
    gather_walker(r, M, w, ne, pos);
    double *out = O + (size_t)w * (size_t)np;
    /* Jastrow: K = a r / (1 + b r)  (D.1):  dK/da = r / (1 + b r),  dK/db = -a r^2 / (1 + b r)^2 */
    real da_par = 0.0, da_anti = 0.0, db = 0.0;
    for (int i = 0; i < ne; ++i)
      for (int j = i + 1; j < ne; ++j) {
        int same = spin_of(s, i) == spin_of(s, j);
        real a = same ? s->jastrow_a_par : s->jastrow_a_anti;
        real dx = pos[3 * i] - pos[3 * j], dy = pos[3 * i + 1] - pos[3 * j + 1], dz = pos[3 * i + 2] - pos[3 * j + 2];
        real rij = sqrt(dx * dx + dy * dy + dz * dz);
        real den = 1.0 + s->jastrow_b * rij;
        if (same) da_par += rij / den; else da_anti += rij / den;
        db += -a * rij * rij / (den * den);
      }
    out[0] = da_par;
    out[1] = da_anti;
    out[2] = db;
    /* electron-nucleus kernel K = (w0 r + w1 r^2) / (1 + w2 r)  (D.2):
     * dK/dw0 = r / D,  dK/dw1 = r^2 / D,  dK/dw2 = -(w0 r + w1 r^2) r / D^2,  D = 1 + w2 r */
    real dw0 = 0.0, dw1 = 0.0, dw2 = 0.0;
    for (int i = 0; i < ne; ++i)
      for (int at = 0; at < s->n_atoms; ++at) {
        real dx = pos[3 * i] - s->atom_xyz[3 * at], dy = pos[3 * i + 1] - s->atom_xyz[3 * at + 1],
               dz = pos[3 * i + 2] - s->atom_xyz[3 * at + 2];
        real ria = sqrt(dx * dx + dy * dy + dz * dz);
        real D = 1.0 + s->jastrow_en_w2 * ria;
        dw0 += ria / D;
        dw1 += ria * ria / D;
        dw2 += -(s->jastrow_en_w0 * ria + s->jastrow_en_w1 * ria * ria) * ria / (D * D);
      }
    out[3] = dw0;
    out[4] = dw1;
    out[5] = dw2;
    /* electron-electron-nucleus kernel (D.3; reading Q22: every nucleus, every pair once and
     * symmetrised = ordered pairs i != j with weight 1/2):
     * term mu = (c/2) f(r_ai) g(r_aj) h(r_ij) with Pade factors p(r) = a r / (1 + b r):
     * dp/da = r / (1 + b r),  dp/db = -a r^2 / (1 + b r)^2.  Seven parameters per term, in the order of
     * een_params: c, a_f, b_f, a_g, b_g, a_h, b_h. */
    for (int mu = 0; mu < s->n_een; ++mu) {
      const double *q = s->een_params + 7 * mu;
      real dq[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
      for (int at = 0; at < s->n_atoms; ++at)
        for (int i = 0; i < ne; ++i)
          for (int j = 0; j < ne; ++j) {
            if (i == j) continue;
            real xi = pos[3 * i] - s->atom_xyz[3 * at], yi = pos[3 * i + 1] - s->atom_xyz[3 * at + 1],
                   zi = pos[3 * i + 2] - s->atom_xyz[3 * at + 2];
            real xj = pos[3 * j] - s->atom_xyz[3 * at], yj = pos[3 * j + 1] - s->atom_xyz[3 * at + 1],
                   zj = pos[3 * j + 2] - s->atom_xyz[3 * at + 2];
            real xx = pos[3 * i] - pos[3 * j], yy = pos[3 * i + 1] - pos[3 * j + 1], zz = pos[3 * i + 2] - pos[3 * j + 2];
            real rai = sqrt(xi * xi + yi * yi + zi * zi), raj = sqrt(xj * xj + yj * yj + zj * zj);
            real rij = sqrt(xx * xx + yy * yy + zz * zz);
            real Df = 1.0 + q[2] * rai, Dg = 1.0 + q[4] * raj, Dh = 1.0 + q[6] * rij;
            real f = q[1] * rai / Df, g = q[3] * raj / Dg, h = q[5] * rij / Dh;
            dq[0] += 0.5 * f * g * h;
            dq[1] += 0.5 * q[0] * (rai / Df) * g * h;
            dq[2] += 0.5 * q[0] * (-q[1] * rai * rai / (Df * Df)) * g * h;
            dq[3] += 0.5 * q[0] * f * (raj / Dg) * h;
            dq[4] += 0.5 * q[0] * f * (-q[3] * raj * raj / (Dg * Dg)) * h;
            dq[5] += 0.5 * q[0] * f * g * (rij / Dh);
            dq[6] += 0.5 * q[0] * f * g * (-q[5] * rij * rij / (Dh * Dh));
          }
      for (int k = 0; k < 7; ++k) out[6 + 7 * mu + k] = dq[k];
    }
    /* CI: Sigma = sum_n d_n D_n^up D_n^dn  (eq. 4):  d ln Sigma / d d_n = D_n^up D_n^dn / Sigma */
    for (int q = 0; q < 3 * ne; ++q) post[q] = pos[q];
    if (bf) backflow_map(s, pos, post, NULL, NULL);
    for (int i = 0; i < ne * nmo; ++i) mo[i] = dmo[i] = 0.0;
    for (int i = 0; i < ne; ++i) {
      real dw[3] = {0.0, 0.0, 0.0};  /* d rt_i / d w */
      for (int j = 0; j < ne; ++j) {
        if (j == i) continue;
        real dx = pos[3 * i] - pos[3 * j], dy = pos[3 * i + 1] - pos[3 * j + 1], dz = pos[3 * i + 2] - pos[3 * j + 2];
        real rij = sqrt(dx * dx + dy * dy + dz * dz);
        dw[0] += dx / rij; dw[1] += dy / rij; dw[2] += dz / rij;
      }
      for (int beta = 0; beta < s->n_ao; ++beta) {
        ao_eval_r(s, beta, post + 3 * i, ao);
        for (int alpha = 0; alpha < nmo; ++alpha) {
          mo[i * nmo + alpha] += s->mo_coeff[beta * nmo + alpha] * ao[0];
          dmo[i * nmo + alpha] += s->mo_coeff[beta * nmo + alpha] * (ao[1] * dw[0] + ao[2] * dw[1] + ao[3] * dw[2]);
        }
      }
    }
    real sigma = 0.0, dsigma = 0.0;
    for (int n = 0; n < s->n_det; ++n) {
      real D[2], tr[2] = {0.0, 0.0};
      for (int sp = 0; sp < 2; ++sp) {
        int ns = sp ? s->n_dn : s->n_up, e0 = sp ? s->n_up : 0;
        const int32_t *lst = sp ? s->det_dn + (size_t)n * s->n_dn : s->det_up + (size_t)n * s->n_up;
        for (int i = 0; i < ns; ++i)
          for (int j = 0; j < ns; ++j) A[i * ns + j] = mo[(e0 + i) * nmo + lst[j]];
        D[sp] = det_inv_r(ns, A, bf ? Ai : NULL);
        if (bf)  /* Tr(A^-1 d_w A) = sum_ij Ai[j][i] d_w A[i][j] */
          for (int i = 0; i < ns; ++i)
            for (int j = 0; j < ns; ++j) tr[sp] += Ai[j * ns + i] * dmo[(e0 + i) * nmo + lst[j]];
      }
      prod[n] = D[0] * D[1];
      sigma += s->ci_coeff[n] * prod[n];
      dsigma += s->ci_coeff[n] * prod[n] * (tr[0] + tr[1]);
    }
    for (int n = 0; n < s->n_det; ++n) out[nj + n] = prod[n] / sigma;
    if (bf) out[nj + s->n_det] = dsigma / sigma;
  }
  free(mo); free(dmo); free(A); free(Ai); free(pos); free(post); free(prod);
  return 0;
}

static double kahan_mean(const double *x, int64_t M) {
  double sum = 0.0, c = 0.0;
  for (int64_t i = 0; i < M; ++i) {
    double y = x[i] - c, t = sum + y;
    c = (t - sum) - y;
    sum = t;
  }
  return sum / (double)M;
}

void oracle_energy_gradient(const double *eloc, const double *O, int64_t M, int32_t n_param,
                            double *Ev, double *grad) {
  double ev = kahan_mean(eloc, M);
  if (Ev) *Ev = ev;
  for (int p = 0; p < n_param; ++p) {
    double sum = 0.0, c = 0.0;
    for (int64_t m = 0; m < M; ++m) {
      double y = O[(size_t)m * (size_t)n_param + p] * (eloc[m] - ev) - c, t = sum + y;
      c = (t - sum) - y;
      sum = t;
    }
    grad[p] = 2.0 * sum / (double)M;
  }
}

/* ------------------------------------------------------------------ */
/* Orbital-parameter derivatives of ln Psi (AO exponents, MO            */
/* coefficients), every determinant inverted explicitly */
/* ------------------------------------------------------------------ */

int oracle_orbital_derivatives(const oracle_system_desc_t *s, const double *r, int64_t M, int64_t w0,
                               int64_t w1, double *dC, double *dzeta) {
  /* With the backflow transformation the orbitals sit at the backflow coordinates rt, which depend on
   * neither C nor zeta: the same formulas with phi and d phi / d zeta evaluated at rt_i. */
  int ne = s->n_up + s->n_dn, nmo = s->n_mo, nao = s->n_ao;
  real *aov = (real *)malloc(sizeof(real) * (size_t)(ne * nao + 1));      /* ao_beta(r_i) */
  real *aoz = (real *)malloc(sizeof(real) * (size_t)(ne * nao + 1));      /* d ao_beta / d zeta (r_i) */
  real *mo = (real *)malloc(sizeof(real) * (size_t)(ne * nmo + 1));
  real *A = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *Ai = (real *)malloc(sizeof(real) * (size_t)(2 * ne * ne + 2));    /* both spins' inverses of one determinant */
  real *gam = (real *)malloc(sizeof(real) * (size_t)(ne * nmo + 1));      /* Gamma[i][alpha], not yet / Sigma */
  real *pos = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  real *pos0 = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  if (!aov || !aoz || !mo || !A || !Ai || !gam || !pos || !pos0) return -1;
  real ao[5];
  for (int64_t w = w0; w < w1; ++w) {
    gather_walker(r, M, w, ne, pos0);
    for (int q = 0; q < 3 * ne; ++q) pos[q] = pos0[q];
    if (s->backflow_w != 0.0) backflow_map(s, pos0, pos, NULL, NULL);  /* pos: where the orbitals are evaluated */
    for (int i = 0; i < ne; ++i)
      for (int beta = 0; beta < nao; ++beta) {
        ao_eval_r(s, beta, pos + 3 * i, ao);
        aov[i * nao + beta] = ao[0];
        /* phi = N S r^k e^{-zeta r}: d phi / d zeta = phi (d ln N / d zeta - r) */
        int at = s->ao_atom[beta];
        real dx = pos[3 * i] - s->atom_xyz[3 * at], dy = pos[3 * i + 1] - s->atom_xyz[3 * at + 1],
               dz = pos[3 * i + 2] - s->atom_xyz[3 * at + 2];
        real rr = sqrt(dx * dx + dy * dy + dz * dz);
        real dlnN = s->ao_norm ? 0.0 : ((real)s->ao_n[beta] + 0.5) / s->ao_zeta[beta];
        aoz[i * nao + beta] = ao[0] * (dlnN - rr);
      }
    for (int i = 0; i < ne * nmo; ++i) { mo[i] = 0.0; gam[i] = 0.0; }
    for (int i = 0; i < ne; ++i)
      for (int beta = 0; beta < nao; ++beta)
        for (int alpha = 0; alpha < nmo; ++alpha) mo[i * nmo + alpha] += s->mo_coeff[beta * nmo + alpha] * aov[i * nao + beta];
    real sigma = 0.0;
    for (int n = 0; n < s->n_det; ++n) {
      real D[2];
      for (int sp = 0; sp < 2; ++sp) {
        int ns = sp ? s->n_dn : s->n_up, e0 = sp ? s->n_up : 0;
        const int32_t *lst = sp ? s->det_dn + (size_t)n * s->n_dn : s->det_up + (size_t)n * s->n_up;
        for (int i = 0; i < ns; ++i)
          for (int j = 0; j < ns; ++j) A[i * ns + j] = mo[(e0 + i) * nmo + lst[j]];
        D[sp] = det_inv_r(ns, A, Ai + sp * ne * ne);
      }
      real wn = s->ci_coeff[n] * D[0] * D[1];
      sigma += wn;
      for (int sp = 0; sp < 2; ++sp) {
        int ns = sp ? s->n_dn : s->n_up, e0 = sp ? s->n_up : 0;
        const int32_t *lst = sp ? s->det_dn + (size_t)n * s->n_dn : s->det_up + (size_t)n * s->n_up;
        const real *inv = Ai + sp * ne * ne;
        /* d ln D / d A[i][j] = A^-1[j][i]; column j of A_n holds MO lst[j] */
        for (int i = 0; i < ns; ++i)
          for (int j = 0; j < ns; ++j) gam[(e0 + i) * nmo + lst[j]] += wn * inv[j * ns + i];
      }
    }
    if (dC)
      for (int beta = 0; beta < nao; ++beta)
        for (int alpha = 0; alpha < nmo; ++alpha) {
          real t = 0.0;
          for (int i = 0; i < ne; ++i) t += aov[i * nao + beta] * gam[i * nmo + alpha];
          dC[((size_t)w * nao + beta) * nmo + alpha] = t / sigma;
        }
    if (dzeta)
      for (int beta = 0; beta < nao; ++beta) {
        real t = 0.0;
        for (int alpha = 0; alpha < nmo; ++alpha) {
          real u = 0.0;
          for (int i = 0; i < ne; ++i) u += aoz[i * nao + beta] * gam[i * nmo + alpha];
          t += s->mo_coeff[beta * nmo + alpha] * u;
        }
        dzeta[(size_t)w * nao + beta] = t / sigma;
      }
  }
  free(aov); free(aoz); free(mo); free(A); free(Ai); free(gam); free(pos); free(pos0);
  return 0;
}

/* ------------------------------------------------------------------ */
/* Nuclear log-gradient of the wavefunction: grad_alpha ln|Psi|, half   */
/* of grad_alpha ln rho in the force estimator (eq. 7). */
/* Every AO of centre a depends on (r_i - R_a) only, so   */
/* d ao_beta(r_i) / d R_a = -grad_r ao_beta(r_i) for beta on a, else 0; */
/* the chain rule through every determinant, inverted explicitly, gives */
/*   d ln Sigma / d R_a = -sum_n w_n sum_{i,j} A_n^-1[j][i]             */
/*                         sum_{beta on a} C[beta][lst_n[j]] grad ao_beta(r_i)  */
/* and the Jastrow kernels that see the nuclei (D.2, D.3) add           */
/*   d K_en(r_ia) / d R_a = -K_en' e_ai,                                 */
/*   d [(c/2) f(r_ai) g(r_aj) h(r_ij)] / d R_a = -(c/2) h (f' g e_ai + f g' e_aj). */
/* The Pade e-e kernel D.1 does not depend on R.                        */
/* ------------------------------------------------------------------ */

int oracle_nuclear_log_gradient(const oracle_system_desc_t *s, const double *r, int64_t M, int64_t w0,
                                int64_t w1, double *dR) {
  /* With the backflow transformation the orbitals sit at the backflow coordinates rt, which do not depend
   * on the nuclei: the Slater part with phi and grad phi at rt_i, the Jastrow parts (at r) unchanged. */
  int ne = s->n_up + s->n_dn, nmo = s->n_mo, nao = s->n_ao, na = s->n_atoms;
  real *aov = (real *)malloc(sizeof(real) * (size_t)(ne * nao + 1));       /* ao_beta(r_i) */
  real *aog = (real *)malloc(sizeof(real) * (size_t)(3 * ne * nao + 1));   /* grad ao_beta(r_i) */
  real *mo = (real *)malloc(sizeof(real) * (size_t)(ne * nmo + 1));
  real *A = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *Ai = (real *)malloc(sizeof(real) * (size_t)(2 * ne * ne + 2));
  real *gam = (real *)malloc(sizeof(real) * (size_t)(ne * nmo + 1));
  real *pos = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  real *post = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  if (!aov || !aog || !mo || !A || !Ai || !gam || !pos || !post) return -1;
  real ao[5];
  for (int64_t w = w0; w < w1; ++w) {
    gather_walker(r, M, w, ne, pos);
    for (int q = 0; q < 3 * ne; ++q) post[q] = pos[q];
    if (s->backflow_w != 0.0) backflow_map(s, pos, post, NULL, NULL);  /* post: where the orbitals are evaluated */
    for (int i = 0; i < ne; ++i)
      for (int beta = 0; beta < nao; ++beta) {
        ao_eval_r(s, beta, post + 3 * i, ao);
        aov[i * nao + beta] = ao[0];
        for (int c = 0; c < 3; ++c) aog[(i * nao + beta) * 3 + c] = ao[1 + c];
      }
    for (int i = 0; i < ne * nmo; ++i) { mo[i] = 0.0; gam[i] = 0.0; }
    for (int i = 0; i < ne; ++i)
      for (int beta = 0; beta < nao; ++beta)
        for (int alpha = 0; alpha < nmo; ++alpha) mo[i * nmo + alpha] += s->mo_coeff[beta * nmo + alpha] * aov[i * nao + beta];
    real sigma = 0.0;
    for (int n = 0; n < s->n_det; ++n) {
      real D[2];
      for (int sp = 0; sp < 2; ++sp) {
        int ns = sp ? s->n_dn : s->n_up, e0 = sp ? s->n_up : 0;
        const int32_t *lst = sp ? s->det_dn + (size_t)n * s->n_dn : s->det_up + (size_t)n * s->n_up;
        for (int i = 0; i < ns; ++i)
          for (int j = 0; j < ns; ++j) A[i * ns + j] = mo[(e0 + i) * nmo + lst[j]];
        D[sp] = det_inv_r(ns, A, Ai + sp * ne * ne);
      }
      real wn = s->ci_coeff[n] * D[0] * D[1];
      sigma += wn;
      for (int sp = 0; sp < 2; ++sp) {
        int ns = sp ? s->n_dn : s->n_up, e0 = sp ? s->n_up : 0;
        const int32_t *lst = sp ? s->det_dn + (size_t)n * s->n_dn : s->det_up + (size_t)n * s->n_up;
        const real *inv = Ai + sp * ne * ne;
        for (int i = 0; i < ns; ++i)
          for (int j = 0; j < ns; ++j) gam[(e0 + i) * nmo + lst[j]] += wn * inv[j * ns + i];
      }
    }
    double *out = dR + (size_t)w * (size_t)(3 * na);
    for (int k = 0; k < 3 * na; ++k) out[k] = 0.0;
    /* Slater part */
    for (int beta = 0; beta < nao; ++beta) {
      int at = s->ao_atom[beta];
      for (int c = 0; c < 3; ++c) {
        real t = 0.0;
        for (int alpha = 0; alpha < nmo; ++alpha) {
          real u = 0.0;
          for (int i = 0; i < ne; ++i) u += aog[(i * nao + beta) * 3 + c] * gam[i * nmo + alpha];
          t += s->mo_coeff[beta * nmo + alpha] * u;
        }
        out[3 * at + c] -= t / sigma;
      }
    }
    /* electron-nucleus kernel D.2: K = N/D, N = w0 r + w1 r^2, D = 1 + w2 r */
    real jw0 = s->jastrow_en_w0, jw1 = s->jastrow_en_w1, jw2 = s->jastrow_en_w2;
    if (jw0 != 0.0 || jw1 != 0.0)
      for (int i = 0; i < ne; ++i)
        for (int at = 0; at < na; ++at) {
          real d[3];
          for (int c = 0; c < 3; ++c) d[c] = pos[3 * i + c] - s->atom_xyz[3 * at + c];
          real ria = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
          real N = jw0 * ria + jw1 * ria * ria, D = 1.0 + jw2 * ria;
          real K1 = ((jw0 + 2.0 * jw1 * ria) * D - N * jw2) / (D * D);
          for (int c = 0; c < 3; ++c) out[3 * at + c] -= K1 * d[c] / ria;
        }
    /* electron-electron-nucleus kernel D.3 (reading Q22: ordered pairs i != j with weight 1/2) */
    for (int at = 0; at < na; ++at)
      for (int i = 0; i < ne; ++i)
        for (int j = 0; j < ne; ++j) {
          if (i == j || s->n_een == 0) continue;
          real eai[3], eaj[3], eij[3];
          for (int c = 0; c < 3; ++c) {
            eai[c] = pos[3 * i + c] - s->atom_xyz[3 * at + c];
            eaj[c] = pos[3 * j + c] - s->atom_xyz[3 * at + c];
            eij[c] = pos[3 * i + c] - pos[3 * j + c];
          }
          real rai = sqrt(eai[0] * eai[0] + eai[1] * eai[1] + eai[2] * eai[2]);
          real raj = sqrt(eaj[0] * eaj[0] + eaj[1] * eaj[1] + eaj[2] * eaj[2]);
          real rij = sqrt(eij[0] * eij[0] + eij[1] * eij[1] + eij[2] * eij[2]);
          for (int mu = 0; mu < s->n_een; ++mu) {
            const double *q = s->een_params + 7 * mu;
            real f, f1, f2, g, g1, g2, h, h1, h2;
            pade3(q[1], q[2], rai, &f, &f1, &f2);
            pade3(q[3], q[4], raj, &g, &g1, &g2);
            pade3(q[5], q[6], rij, &h, &h1, &h2);
            for (int c = 0; c < 3; ++c)
              out[3 * at + c] -= 0.5 * q[0] * h * (f1 * g * eai[c] / rai + f * g1 * eaj[c] / raj);
          }
        }
  }
  free(aov); free(aog); free(mo); free(A); free(Ai); free(gam); free(pos); free(post);
  return 0;
}

/* ------------------------------------------------------------------ */
/* Second-level AO derivatives for the forces (eq. 7):    */
/* the atomic positions are inputs of the AO layer,  */
/* d ao(r_i) / d R = -grad_r ao(r_i), so grad_R E_L needs the Hessian  */
/* of every AO and the gradient of its Laplacian.  Product rule term   */
/* by term on phi = N S(d) f(r), f = r^k e^{-zeta r}, u = d / r:        */
/*  d_c d_e phi = N [S_ce f + (S_c u_e + S_e u_c) f' + S (f'' u_c u_e  */
/*                   + f' (delta_ce - u_c u_e) / r)]                    */
/*  lap phi     = N [lapS f + 2 f' (grad S . u) + S (f'' + 2 f'/r)]     */
/*  d_c lap phi = N [lapS f' u_c + 2 f'' u_c (grad S . u)               */
/*                   + 2 f' d_c(grad S . u) + S_c (f'' + 2 f'/r)        */
/*                   + S (f''' + 2 f''/r - 2 f'/r^2) u_c]               */
/*  d_c (grad S . u) = sum_e [S_ec u_e + S_e (delta_ec - u_e u_c) / r]  */
/* out14 = {phi, grad[3], lap, hess xx yy zz xy yz zx, grad lap[3]}    */
/* ------------------------------------------------------------------ */

static void solid_harmonic_hessian(int l, int m, real H[3][3]) {
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) H[a][b] = 0.0;
  if (l != 2) return; /* S is constant or linear */
  if (m == 0) H[0][1] = H[1][0] = 1.0;                          /* xy */
  if (m == 1) H[1][2] = H[2][1] = 1.0;                          /* yz */
  if (m == 2) H[0][2] = H[2][0] = 1.0;                          /* zx */
  if (m == 3) { H[0][0] = 2.0; H[1][1] = -2.0; }                /* x^2 - y^2 */
  if (m == 4) { H[0][0] = -2.0; H[1][1] = -2.0; H[2][2] = 4.0; } /* 2 z^2 - x^2 - y^2 */
}

static void ao_eval2_r(const oracle_system_desc_t *s, int ao, const real *xyz, real *out14) {
  int a = s->ao_atom[ao], n = s->ao_n[ao], l = s->ao_l[ao], m = s->ao_m[ao];
  real zeta = s->ao_zeta[ao];
  real N = s->ao_norm ? s->ao_norm[ao] : sto_norm_r(n, l, m, zeta);
  real d[3], u[3];
  for (int c = 0; c < 3; ++c) d[c] = xyz[c] - s->atom_xyz[3 * a + c];
  real r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
  for (int c = 0; c < 3; ++c) u[c] = d[c] / r;
  int k = n - 1 - l;
  real S, gS[3], hS[3], HS[3][3];
  solid_harmonic(l, m, d[0], d[1], d[2], &S, gS, hS);
  solid_harmonic_hessian(l, m, HS);
  real lapS = HS[0][0] + HS[1][1] + HS[2][2];
  /* radial factor and three derivatives, term by term */
  real e = exp(-zeta * r);
  real rk = pow(r, (real)k);
  real rk1 = (k >= 1) ? pow(r, (real)(k - 1)) : 0.0;
  real rk2 = (k >= 2) ? pow(r, (real)(k - 2)) : 0.0;
  real rk3 = (k >= 3) ? pow(r, (real)(k - 3)) : 0.0;
  real f = rk * e;
  real f1 = ((real)k * rk1 - zeta * rk) * e;
  real f2 = ((real)(k * (k - 1)) * rk2 - 2.0 * (real)k * zeta * rk1 + zeta * zeta * rk) * e;
  real f3 = ((real)(k * (k - 1) * (k - 2)) * rk3 - 3.0 * (real)(k * (k - 1)) * zeta * rk2 + 3.0 * (real)k * zeta * zeta * rk1 -
             zeta * zeta * zeta * rk) * e;
  real gSu = gS[0] * u[0] + gS[1] * u[1] + gS[2] * u[2];
  out14[0] = N * S * f;
  for (int c = 0; c < 3; ++c) out14[1 + c] = N * (gS[c] * f + S * f1 * u[c]);
  out14[4] = N * (lapS * f + 2.0 * f1 * gSu + S * (f2 + 2.0 * f1 / r));
  real hess[3][3];
  for (int c = 0; c < 3; ++c)
    for (int q = 0; q < 3; ++q) {
      real dl = (c == q) ? 1.0 : 0.0;
      hess[c][q] = N * (HS[c][q] * f + (gS[c] * u[q] + gS[q] * u[c]) * f1 + S * (f2 * u[c] * u[q] + f1 * (dl - u[c] * u[q]) / r));
    }
  out14[5] = hess[0][0]; out14[6] = hess[1][1]; out14[7] = hess[2][2];
  out14[8] = hess[0][1]; out14[9] = hess[1][2]; out14[10] = hess[2][0];
  for (int c = 0; c < 3; ++c) {
    real dgSu = 0.0;
    for (int q = 0; q < 3; ++q) dgSu += HS[q][c] * u[q] + gS[q] * (((q == c) ? 1.0 : 0.0) - u[q] * u[c]) / r;
    out14[11 + c] = N * (lapS * f1 * u[c] + 2.0 * f2 * u[c] * gSu + 2.0 * f1 * dgSu + gS[c] * (f2 + 2.0 * f1 / r) +
                         S * (f3 + 2.0 * f2 / r - 2.0 * f1 / (r * r)) * u[c]);
  }
}

void oracle_ao_eval2(const oracle_system_desc_t *s, int ao, const double *xyz, double *out14) {
  real p[3] = {xyz[0], xyz[1], xyz[2]}, o[14];
  ao_eval2_r(s, ao, p, o);
  for (int q = 0; q < 14; ++q) out14[q] = (double)o[q];
}

/* ------------------------------------------------------------------ */
/* grad_alpha E_L, the first term of the force estimator (eq. 7,       */
/* PAPER.md:86), for the Pade e-e Jastrow D.1 (which does not see the  */
/* nuclei).  Differentiates, long-hand, exactly what local_energy_one  */
/* evaluates:                                                           */
/*   E_L = -1/2 [lapJ + |gJ|^2 + 2 gJ . gS / S + lapS / S] + V          */
/*   S = sum_n w_n, w_n = d_n D_n^up D_n^dn; gS = sum_n w_n gamma_n,     */
/*   gamma_n[i] = sum_k A^-1[k][i] grad phi_k(r_i) (F.3 / G.2);          */
/*   lapS = sum_n w_n t_n, t_n = sum_ik A^-1[k][i] lap phi_k(r_i) (G.7)  */
/* with, for a displacement of R_alpha,c (written d_j below):            */
/*   d_j A[i][k] = -sum_{beta on alpha} C[beta][k] d_c ao_beta(r_i)      */
/*   d_j ln D = Tr(A^-1 d_j A),  d_j A^-1 = -A^-1 (d_j A) A^-1           */
/*   d_j w_n = w_n (Tr^up + Tr^dn)                                       */
/* and the same chain rule on gamma_n and t_n (AO Hessian, gradient of   */
/* the AO Laplacian), every determinant inverted explicitly.  The        */
/* potential adds  d V_en / d R_alpha = -Z_alpha sum_i (r_i - R_alpha) / */
/* |r_i - R_alpha|^3  and  d V_nn / d R_alpha = -Z_alpha sum_beta Z_beta */
/* (R_alpha - R_beta) / |R_alpha - R_beta|^3   (eq. 1).     */
/* dE [M][n_atoms][3].  Returns -2 when the wavefunction carries the     */
/* e-n / e-e-n Jastrow kernels (their R-dependence is not derived here). */
/* ------------------------------------------------------------------ */

int oracle_nuclear_energy_gradient(const oracle_system_desc_t *s, const double *r, int64_t M, int64_t w0,
                                   int64_t w1, double *dE) {
  if (s->jastrow_en_w0 != 0.0 || s->jastrow_en_w1 != 0.0 || s->n_een > 0 || s->backflow_w != 0.0) return -2;
  int ne = s->n_up + s->n_dn, nmo = s->n_mo, nao = s->n_ao, na = s->n_atoms, nj = 3 * na;
  size_t nem = (size_t)ne * (size_t)nmo;
  real *mo = (real *)malloc(sizeof(real) * (nem * 5 + 1));                 /* [i][a]{val, gx, gy, gz, lap} */
  real *dval = (real *)malloc(sizeof(real) * ((size_t)nj * nem + 1));       /* d_j phi_a(r_i) */
  real *dgrd = (real *)malloc(sizeof(real) * ((size_t)nj * nem * 3 + 1));   /* d_j d_q phi_a(r_i) */
  real *dlap = (real *)malloc(sizeof(real) * ((size_t)nj * nem + 1));       /* d_j lap phi_a(r_i) */
  real *A = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *Ai = (real *)malloc(sizeof(real) * (size_t)(2 * ne * ne + 2));
  real *dA = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *dAi = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *tmp = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *gam = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));          /* gamma_n of the current determinant */
  real *dgam = (real *)malloc(sizeof(real) * (size_t)(nj * 3 * ne + 1));    /* d_j gamma_n */
  real *gS = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  real *dgS = (real *)malloc(sizeof(real) * (size_t)(nj * 3 * ne + 1));
  real *gJ = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  real *pos = (real *)malloc(sizeof(real) * (size_t)(3 * ne + 1));
  real *tr = (real *)malloc(sizeof(real) * (size_t)(2 * nj + 1));
  real *dt = (real *)malloc(sizeof(real) * (size_t)(2 * nj + 1));
  real *dSig = (real *)malloc(sizeof(real) * (size_t)(nj + 1));
  real *dlapS = (real *)malloc(sizeof(real) * (size_t)(nj + 1));
  if (!mo || !dval || !dgrd || !dlap || !A || !Ai || !dA || !dAi || !tmp || !gam || !dgam || !gS || !dgS || !gJ || !pos ||
      !tr || !dt || !dSig || !dlapS)
    return -1;
  real ao[14];
  for (int64_t w = w0; w < w1; ++w) {
    gather_walker(r, M, w, ne, pos);
    for (size_t q = 0; q < nem * 5; ++q) mo[q] = 0.0;
    for (size_t q = 0; q < (size_t)nj * nem; ++q) { dval[q] = 0.0; dlap[q] = 0.0; }
    for (size_t q = 0; q < (size_t)nj * nem * 3; ++q) dgrd[q] = 0.0;
    for (int i = 0; i < ne; ++i)
      for (int beta = 0; beta < nao; ++beta) {
        ao_eval2_r(s, beta, pos + 3 * i, ao);
        int at = s->ao_atom[beta];
        real hess[3][3] = {{ao[5], ao[8], ao[10]}, {ao[8], ao[6], ao[9]}, {ao[10], ao[9], ao[7]}};
        for (int a = 0; a < nmo; ++a) {
          real cf = s->mo_coeff[beta * nmo + a];
          for (int q = 0; q < 5; ++q) mo[((size_t)i * nmo + a) * 5 + q] += cf * ao[q];
          for (int c = 0; c < 3; ++c) { /* d / d R_{at,c} = - d / d r_c on this AO */
            size_t j = (size_t)(3 * at + c);
            dval[j * nem + (size_t)i * nmo + a] -= cf * ao[1 + c];
            for (int q = 0; q < 3; ++q) dgrd[(j * nem + (size_t)i * nmo + a) * 3 + q] -= cf * hess[c][q];
            dlap[j * nem + (size_t)i * nmo + a] -= cf * ao[11 + c];
          }
        }
      }
    real J, lapJ;
    jastrow_all(s, pos, &J, gJ, &lapJ);
    real sigma = 0.0, lapS = 0.0;
    for (int i = 0; i < 3 * ne; ++i) gS[i] = 0.0;
    for (int j = 0; j < nj; ++j) { dSig[j] = 0.0; dlapS[j] = 0.0; }
    for (int q = 0; q < nj * 3 * ne; ++q) dgS[q] = 0.0;
    for (int n = 0; n < s->n_det; ++n) {
      real D[2], t[2];
      for (int sp = 0; sp < 2; ++sp) {
        int ns = sp ? s->n_dn : s->n_up, e0 = sp ? s->n_up : 0;
        const int32_t *lst = sp ? s->det_dn + (size_t)n * s->n_dn : s->det_up + (size_t)n * s->n_up;
        real *inv = Ai + sp * ne * ne;
        for (int i = 0; i < ns; ++i)
          for (int k = 0; k < ns; ++k) A[i * ns + k] = mo[((size_t)(e0 + i) * nmo + lst[k]) * 5 + 0];
        D[sp] = det_inv_r(ns, A, inv);
        t[sp] = 0.0;
        for (int i = 0; i < ns; ++i) {
          for (int c = 0; c < 3; ++c) {
            real g = 0.0;
            for (int k = 0; k < ns; ++k) g += inv[k * ns + i] * mo[((size_t)(e0 + i) * nmo + lst[k]) * 5 + 1 + c];
            gam[3 * (e0 + i) + c] = g;
          }
          for (int k = 0; k < ns; ++k) t[sp] += inv[k * ns + i] * mo[((size_t)(e0 + i) * nmo + lst[k]) * 5 + 4];
        }
        for (int j = 0; j < nj; ++j) {
          const real *dv = dval + (size_t)j * nem, *dg = dgrd + (size_t)j * nem * 3, *dl = dlap + (size_t)j * nem;
          for (int i = 0; i < ns; ++i)
            for (int k = 0; k < ns; ++k) dA[i * ns + k] = dv[(size_t)(e0 + i) * nmo + lst[k]];
          real trj = 0.0;
          for (int i = 0; i < ns; ++i)
            for (int k = 0; k < ns; ++k) trj += inv[k * ns + i] * dA[i * ns + k];
          tr[2 * j + sp] = trj;
          /* d A^-1 = -A^-1 dA A^-1 */
          for (int i = 0; i < ns; ++i)
            for (int k = 0; k < ns; ++k) {
              real v = 0.0;
              for (int q = 0; q < ns; ++q) v += dA[i * ns + q] * inv[q * ns + k];
              tmp[i * ns + k] = v;
            }
          for (int i = 0; i < ns; ++i)
            for (int k = 0; k < ns; ++k) {
              real v = 0.0;
              for (int q = 0; q < ns; ++q) v += inv[i * ns + q] * tmp[q * ns + k];
              dAi[i * ns + k] = -v;
            }
          real dtj = 0.0;
          for (int i = 0; i < ns; ++i) {
            for (int c = 0; c < 3; ++c) {
              real g = 0.0;
              for (int k = 0; k < ns; ++k)
                g += dAi[k * ns + i] * mo[((size_t)(e0 + i) * nmo + lst[k]) * 5 + 1 + c] +
                     inv[k * ns + i] * dg[((size_t)(e0 + i) * nmo + lst[k]) * 3 + c];
              dgam[(j * ne + e0 + i) * 3 + c] = g;
            }
            for (int k = 0; k < ns; ++k)
              dtj += dAi[k * ns + i] * mo[((size_t)(e0 + i) * nmo + lst[k]) * 5 + 4] + inv[k * ns + i] * dl[(size_t)(e0 + i) * nmo + lst[k]];
          }
          dt[2 * j + sp] = dtj;
        }
      }
      real wn = s->ci_coeff[n] * D[0] * D[1];
      sigma += wn;
      for (int i = 0; i < 3 * ne; ++i) gS[i] += wn * gam[i];
      lapS += wn * (t[0] + t[1]);
      for (int j = 0; j < nj; ++j) {
        real dw = wn * (tr[2 * j] + tr[2 * j + 1]);
        dSig[j] += dw;
        for (int i = 0; i < 3 * ne; ++i) dgS[j * 3 * ne + i] += dw * gam[i] + wn * dgam[j * 3 * ne + i];
        dlapS[j] += dw * (t[0] + t[1]) + wn * (dt[2 * j] + dt[2 * j + 1]);
      }
    }
    double *out = dE + (size_t)w * (size_t)nj;
    for (int at = 0; at < na; ++at)
      for (int c = 0; c < 3; ++c) {
        int j = 3 * at + c;
        /* kinetic: -1/2 [2 gJ . d(gS/S) + d(lapS/S)] */
        real cross = 0.0;
        for (int i = 0; i < 3 * ne; ++i) cross += gJ[i] * (dgS[j * 3 * ne + i] / sigma - gS[i] * dSig[j] / (sigma * sigma));
        real dkin = -0.5 * (2.0 * cross + dlapS[j] / sigma - lapS * dSig[j] / (sigma * sigma));
        /* potential */
        real dven = 0.0, dvnn = 0.0;
        for (int i = 0; i < ne; ++i) {
          real dx = pos[3 * i] - s->atom_xyz[3 * at], dy = pos[3 * i + 1] - s->atom_xyz[3 * at + 1],
               dz = pos[3 * i + 2] - s->atom_xyz[3 * at + 2];
          real rho = sqrt(dx * dx + dy * dy + dz * dz);
          real dc = (c == 0) ? dx : ((c == 1) ? dy : dz);
          dven -= s->atom_Z[at] * dc / (rho * rho * rho);
        }
        for (int b = 0; b < na; ++b) {
          if (b == at) continue;
          real dx = s->atom_xyz[3 * at] - s->atom_xyz[3 * b], dy = s->atom_xyz[3 * at + 1] - s->atom_xyz[3 * b + 1],
               dz = s->atom_xyz[3 * at + 2] - s->atom_xyz[3 * b + 2];
          real rho = sqrt(dx * dx + dy * dy + dz * dz);
          real dc = (c == 0) ? dx : ((c == 1) ? dy : dz);
          dvnn -= s->atom_Z[at] * s->atom_Z[b] * dc / (rho * rho * rho);
        }
        out[j] = (double)(dkin + dven + dvnn);
      }
  }
  free(mo); free(dval); free(dgrd); free(dlap); free(A); free(Ai); free(dA); free(dAi); free(tmp); free(gam); free(dgam);
  free(gS); free(dgS); free(gJ); free(pos); free(tr); free(dt); free(dSig); free(dlapS);
  return 0;
}

/* ------------------------------------------------------------------ */
/* Force estimator, eq. 7 (reading Q23: the minus sign     */
/* covers both terms, ln rho = 2 ln|Psi|):                              */
/*   F_alpha = -(1/M) sum_m [grad_alpha E_L + 2 (E_L - E_v) grad_alpha ln|Psi|] */
/* Kahan sums.  F [n_atoms][3]; terms [2][n_atoms][3] (may be NULL)     */
/* receives the two contributions separately.                           */
/* ------------------------------------------------------------------ */

void oracle_force(const double *eloc, const double *dE, const double *dlnpsi, int64_t M, int32_t n_atoms,
                  double *F, double *terms) {
  double ev = kahan_mean(eloc, M);
  for (int j = 0; j < 3 * n_atoms; ++j) {
    double s1 = 0.0, c1 = 0.0, s2 = 0.0, c2 = 0.0;
    for (int64_t m = 0; m < M; ++m) {
      double y = dE[(size_t)m * (size_t)(3 * n_atoms) + j] - c1, t = s1 + y;
      c1 = (t - s1) - y;
      s1 = t;
      y = 2.0 * (eloc[m] - ev) * dlnpsi[(size_t)m * (size_t)(3 * n_atoms) + j] - c2;
      t = s2 + y;
      c2 = (t - s2) - y;
      s2 = t;
    }
    double a = -s1 / (double)M, b = -s2 / (double)M;
    F[j] = a + b;
    if (terms) { terms[j] = a; terms[3 * n_atoms + j] = b; }
  }
}


/* ------------------------------------------------------------------ */
/* Local energy of a backflow-transformed wavefunction (PAPER.md:53;    */
/* F.1, F.2, F.4 with its cross term, F.3, F.5).       */
/* The plain definition, coordinate by coordinate: for each of the 3 N_e */
/* electron coordinates x_l the dense derivative matrices                */
/*   (d_l A)[i][k]   = sum_a d_a phi_k(rt_i) J[i][a][l]                   */
/*   (d_l^2 A)[i][k] = sum_aa' H_aa' phi_k(rt_i) J[i][a][l] J[i][a'][l]   */
/*                     + sum_a d_a phi_k(rt_i) d^2 rt_i^a / d x_l^2        */
/* (J = Jacobian of the backflow map) and for every determinant and spin */
/*   d_l D / D     = Tr(A^-1 d_l A)                                (F.3)  */
/*   d_l^2 D / D   = Tr(A^-1 d_l^2 A) + Tr(A^-1 d_l A)^2                  */
/*                   - Tr(A^-1 d_l A A^-1 d_l A)                   (F.5)  */
/*   grad Sigma    = sum_n w_n (grad D^up/D^up + grad D^dn/D^dn)   (F.2)  */
/*   lap Sigma     = sum_n w_n (lap D^up/D^up + 2 grad D^up/D^up . grad   */
/*                   D^dn/D^dn + lap D^dn/D^dn)                    (F.4)  */
/* then F.1 and eq. 1 as in local_energy_one.                            */
/* ------------------------------------------------------------------ */
static void local_energy_backflow_one(const oracle_system_desc_t *s, const real *r, real *logpsi, real *sign, real *eloc,
                                      real *parts) {
  int ne = s->n_up + s->n_dn, nmo = s->n_mo, nc = 3 * ne;
  size_t nem = (size_t)ne * (size_t)nmo;
  real *rt = (real *)malloc(sizeof(real) * (size_t)(nc + 1));
  real *jac = (real *)malloc(sizeof(real) * (size_t)(ne * 3 * nc + 1));
  real *lap2 = (real *)malloc(sizeof(real) * (size_t)(ne * 3 * nc + 1));
  real *mo = (real *)malloc(sizeof(real) * (nem * 10 + 1));  /* [i][k]{val, gx, gy, gz, hxx, hyy, hzz, hxy, hyz, hzx} */
  real *dA = (real *)malloc(sizeof(real) * ((size_t)nc * nem + 1));   /* [l][i][k] first derivative of the MO matrix */
  real *d2A = (real *)malloc(sizeof(real) * ((size_t)nc * nem + 1));  /* [l][i][k] second */
  real *A = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *Ai = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *G = (real *)malloc(sizeof(real) * (size_t)(ne * ne + 1));
  real *gJ = (real *)malloc(sizeof(real) * (size_t)(nc + 1));
  real *gS = (real *)malloc(sizeof(real) * (size_t)(nc + 1));
  real *tr1 = (real *)malloc(sizeof(real) * (size_t)(2 * nc + 1));
  backflow_map(s, r, rt, jac, lap2);
  real ao[14];
  for (size_t q = 0; q < nem * 10; ++q) mo[q] = 0.0;
  for (int i = 0; i < ne; ++i)
    for (int beta = 0; beta < s->n_ao; ++beta) {
      ao_eval2_r(s, beta, rt + 3 * i, ao);
      for (int k = 0; k < nmo; ++k) {
        real cf = s->mo_coeff[beta * nmo + k];
        real *m = mo + ((size_t)i * nmo + k) * 10;
        m[0] += cf * ao[0];
        for (int a = 0; a < 3; ++a) m[1 + a] += cf * ao[1 + a];
        for (int q = 0; q < 6; ++q) m[4 + q] += cf * ao[5 + q];
      }
    }
  for (int l = 0; l < nc; ++l)
    for (int i = 0; i < ne; ++i)
      for (int k = 0; k < nmo; ++k) {
        const real *m = mo + ((size_t)i * nmo + k) * 10;
        real H[3][3] = {{m[4], m[7], m[9]}, {m[7], m[5], m[8]}, {m[9], m[8], m[6]}};
        real d1 = 0.0, d2 = 0.0;
        for (int a = 0; a < 3; ++a) {
          real ja = jac[(3 * i + a) * nc + l];
          d1 += m[1 + a] * ja;
          d2 += m[1 + a] * lap2[(3 * i + a) * nc + l];
          for (int b = 0; b < 3; ++b) d2 += H[a][b] * ja * jac[(3 * i + b) * nc + l];
        }
        dA[(size_t)l * nem + (size_t)i * nmo + k] = d1;
        d2A[(size_t)l * nem + (size_t)i * nmo + k] = d2;
      }
  real J, lapJ;
  jastrow_all(s, r, &J, gJ, &lapJ);
  real sigma = 0.0, lapS = 0.0;
  for (int l = 0; l < nc; ++l) gS[l] = 0.0;
  for (int n = 0; n < s->n_det; ++n) {
    real D[2], lapD[2];
    for (int sp = 0; sp < 2; ++sp) {
      int ns = sp ? s->n_dn : s->n_up, e0 = sp ? s->n_up : 0;
      const int32_t *lst = sp ? s->det_dn + (size_t)n * s->n_dn : s->det_up + (size_t)n * s->n_up;
      for (int i = 0; i < ns; ++i)
        for (int k = 0; k < ns; ++k) A[i * ns + k] = mo[((size_t)(e0 + i) * nmo + lst[k]) * 10];
      D[sp] = det_inv_r(ns, A, Ai);
      lapD[sp] = 0.0;
      for (int l = 0; l < nc; ++l) {
        const real *d1 = dA + (size_t)l * nem, *d2 = d2A + (size_t)l * nem;
        /* G = A^-1 d_l A  (orbital positions x orbital positions) */
        real t1 = 0.0, t2 = 0.0, tl = 0.0;
        for (int p = 0; p < ns; ++p)
          for (int q = 0; q < ns; ++q) {
            real v = 0.0, u = 0.0;
            for (int i = 0; i < ns; ++i) {
              v += Ai[p * ns + i] * d1[(size_t)(e0 + i) * nmo + lst[q]];
              if (p == q) u += Ai[p * ns + i] * d2[(size_t)(e0 + i) * nmo + lst[q]];
            }
            G[p * ns + q] = v;
            if (p == q) { t1 += v; tl += u; }
          }
        for (int p = 0; p < ns; ++p)
          for (int q = 0; q < ns; ++q) t2 += G[p * ns + q] * G[q * ns + p];
        tr1[sp * nc + l] = t1;                 /* F.3 */
        lapD[sp] += tl + t1 * t1 - t2;         /* F.5 */
      }
    }
    real wn = s->ci_coeff[n] * D[0] * D[1];
    real cross = 0.0;
    for (int l = 0; l < nc; ++l) cross += tr1[l] * tr1[nc + l];
    sigma += wn;
    for (int l = 0; l < nc; ++l) gS[l] += wn * (tr1[l] + tr1[nc + l]);   /* F.2 */
    lapS += wn * (lapD[0] + 2.0 * cross + lapD[1]);                      /* F.4 */
  }
  real gJ2 = 0.0, crossJ = 0.0;
  for (int l = 0; l < nc; ++l) { gJ2 += gJ[l] * gJ[l]; crossJ += gJ[l] * gS[l]; }
  real kinetic = -0.5 * (lapJ + gJ2 + 2.0 * crossJ / sigma + lapS / sigma);   /* F.1 */
  real vee = 0.0, ven = 0.0, vnn = 0.0;
  for (int i = 0; i < ne; ++i)
    for (int j = i + 1; j < ne; ++j) {
      real dx = r[3 * i] - r[3 * j], dy = r[3 * i + 1] - r[3 * j + 1], dz = r[3 * i + 2] - r[3 * j + 2];
      vee += 1.0 / sqrt(dx * dx + dy * dy + dz * dz);
    }
  for (int i = 0; i < ne; ++i)
    for (int a = 0; a < s->n_atoms; ++a) {
      real dx = r[3 * i] - s->atom_xyz[3 * a], dy = r[3 * i + 1] - s->atom_xyz[3 * a + 1], dz = r[3 * i + 2] - s->atom_xyz[3 * a + 2];
      ven -= s->atom_Z[a] / sqrt(dx * dx + dy * dy + dz * dz);
    }
  for (int a = 0; a < s->n_atoms; ++a)
    for (int b = a + 1; b < s->n_atoms; ++b) {
      real dx = s->atom_xyz[3 * a] - s->atom_xyz[3 * b], dy = s->atom_xyz[3 * a + 1] - s->atom_xyz[3 * b + 1],
           dz = s->atom_xyz[3 * a + 2] - s->atom_xyz[3 * b + 2];
      vnn += s->atom_Z[a] * s->atom_Z[b] / sqrt(dx * dx + dy * dy + dz * dz);
    }
  *logpsi = J + log(fabs(sigma));
  *sign = (sigma > 0.0) ? 1.0 : ((sigma < 0.0) ? -1.0 : 0.0);
  *eloc = kinetic + vee + ven + vnn;
  if (parts) { parts[0] = kinetic; parts[1] = vee; parts[2] = ven; parts[3] = vnn; }
  free(rt); free(jac); free(lap2); free(mo); free(dA); free(d2A); free(A); free(Ai); free(G); free(gJ); free(gS); free(tr1);
}
