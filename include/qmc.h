/* qmc.h -- C ABI of libqmcb200: batched Slater-Jastrow Psi, local energy and
 * all-electron Metropolis sampling in FP64 on one B200 (sm_100a).
 *
 * The calls follow the paper's statement of the problem
 * (/root/reference/PAPER.md, cited as PAPER.md:<line>):
 *   Psi(r) = e^{J(r)} * sum_n d_n D_n^up(r^up) D_n^dn(r^dn)           eq. 4
 *   E_L(r) = H Psi / Psi with the molecular Hamiltonian of eq. 1
 *   walkers sampled from |Psi|^2 by Metropolis-Hastings, all electrons
 *   moved at once with a normal proposal
 *
 * Conventions
 *  - "host" / "device" is stated for every pointer.  The caller owns every
 *    walker / output buffer; a qmc_system_t owns device copies of the
 *    constants given to qmc_setup, which are immutable afterwards, and small
 *    scratch buffers: one per calling stream for the explicit fallback of
 *    qmc_local_energy (grown on demand under a mutex), so calls on different
 *    streams may run concurrently, and the double buffers of
 *    qmc_local_energy_host (one such call at a time per handle).
 *  - qmc_local_energy, qmc_log_psi, qmc_log_derivatives and qmc_metropolis
 *    (without d_eloc_acc and h_n_accepted) make no allocation once a call of
 *    the same size has been made on the stream, and can then be captured in
 *    a CUDA graph.
 *  - Walker coordinates are SoA: double r[n_e][3][M], walker index fastest,
 *    electrons 0..n_up-1 spin-up, the rest spin-down, units bohr.
 *  - Every call returns QMC_OK (0) or a negative status; nothing aborts or
 *    prints.  qmc_status_string(status) describes it; for QMC_ECUDA it carries
 *    the CUDA error text of the failing call on this thread.
 *  - Calls are asynchronous on `cuda_stream` (a cudaStream_t passed as void*)
 *    unless a host out-pointer is given, in which case the call synchronises
 *    that stream before returning.
 *  - There is no CPU fallback: without a CUDA device every call fails with
 *    QMC_ECUDA.
 */
#ifndef QMC_B200_H
#define QMC_B200_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QMC_OK 0
#define QMC_EINVAL (-1)       /* bad argument (null pointer, M <= 0, bad AO quantum numbers, ...) */
#define QMC_EUNSUPPORTED (-2) /* valid problem outside the compiled limits (see qmc_setup) */
#define QMC_ECUDA (-3)        /* a CUDA runtime call failed */
#define QMC_ENOMEM (-4)       /* host allocation failed */
#define QMC_ETOOLARGE (-5)    /* size beyond the fixed scratch of the allocation-free entry point */

typedef struct qmc_system qmc_system_t; /* opaque */

/* Inputs of eq. 4.  All pointers are HOST pointers; the
 * arrays are copied during qmc_setup and may be freed afterwards. */
typedef struct {
  int32_t n_atoms;
  const double *atom_xyz; /* [n_atoms][3] nuclear positions R_alpha, bohr          (eq. 1) */
  const double *atom_Z;   /* [n_atoms] nuclear charges Z_alpha                      (eq. 1) */
  int32_t n_up, n_dn;     /* electrons per spin; n_up + n_dn >= 1 */
  /* Slater-type atomic orbitals:
   *   phi = N * S_lm(d) * r^(n-1-l) * exp(-zeta r),  d = r_i - R_atom, r = |d|,
   * S_lm real solid harmonics, m index:  l=0: {1};  l=1: {x, y, z};
   *   l=2: {xy, yz, zx, x^2-y^2, 2z^2-x^2-y^2}.   Requires 1 <= n <= 4, 0 <= l <= 2, l < n. */
  int32_t n_ao;
  const int32_t *ao_atom; /* [n_ao] centre index */
  const int32_t *ao_n;    /* [n_ao] principal quantum number */
  const int32_t *ao_l;    /* [n_ao] */
  const int32_t *ao_m;    /* [n_ao] harmonic index within l (see above) */
  const double *ao_zeta;  /* [n_ao] exponents, > 0 */
  const double *ao_norm;  /* [n_ao] normalisation N, or NULL for the standard one:
                             (2 zeta)^(n+1/2)/sqrt((2n)!) times the real-spherical-harmonic constant */
  /* Molecular orbitals: phi_alpha = sum_beta C[beta][alpha] ao_beta,
   * C = c * mu already multiplied by the caller. */
  int32_t n_mo;
  const double *mo_coeff; /* [n_ao][n_mo] row-major */
  /* CI expansion: determinant n uses, for each spin, the ORDERED list of
   * MO columns det_x[n][0..n_x-1]:  A_n[i][j] = phi_{det[n][j]}(r_i)  (rows = electrons).
   * Determinant 0 is the reference; the others are usually in-place substitutions of
   * its columns, any number of substitutions is accepted. */
  int32_t n_det;
  const int32_t *det_up; /* [n_det][n_up] (ignored when n_up == 0) */
  const int32_t *det_dn; /* [n_det][n_dn] (ignored when n_dn == 0) */
  const double *ci_coeff; /* [n_det] d_n */
  /* Pade electron-electron Jastrow (D.1): K(r) = w0 r / (1 + w r) */
  double jastrow_a_par;  /* w0 for parallel spins      (cusp value 1/4) */
  double jastrow_a_anti; /* w0 for anti-parallel spins (cusp value 1/2) */
  double jastrow_b;      /* w */
  /* Electron-nucleus Jastrow kernel (D.2), summed over every
   * (electron, nucleus) pair with one parameter set: K_en(r) = (w0 r + w1 r^2) / (1 + w2 r).
   * w0 = w1 = 0 switches the term off. */
  double jastrow_en_w0, jastrow_en_w1, jastrow_en_w2;
  /* Electron-electron-nucleus Jastrow kernel (D.3): n_een terms (at most 6; the paper uses 5),
   * een_params host [n_een][7] = (c, a1, b1, a2, b2, a3, b3) per term:
   *   K_een = sum_mu c [a1 r_ai / (1 + b1 r_ai)] [a2 r_aj / (1 + b2 r_aj)] [a3 r_ij / (1 + b3 r_ij)],
   * summed as eq. 5 says (sum over alpha and i > j, every nucleus, every electron pair once), each pair
   * symmetrised: 1/2 [K_een(r_ai, r_aj, r_ij) + K_een(r_aj, r_ai, r_ij)].  With a1 = a2, b1 = b2 this is the paper's
   * literal sum; with different first and second factors the literal K_een is not symmetric in (i, j) and would break
   * the exchange symmetry of PAPER.md:51, the symmetrised pair does not (reading Q22).  n_een = 0: absent. */
  int32_t n_een;
  const double *een_params;
  /* Inverse backflow transformation (PAPER.md:53 with the kernel of PAPER.md:97):
   *   rt_i = r_i + sum_{j != i} K_BF(r_ij) (r_i - r_j),  K_BF(r) = backflow_w / r,  over all other electrons.
   * The orbitals are evaluated at rt, the Jastrow factor at r.  0 = no backflow.  With backflow on, qmc_local_energy
   * (and the E_L of qmc_metropolis' d_eloc_acc) evaluates the general formulas F.4 / F.5: from
   * the reference determinant's tables (F.6-F.9) when no determinant substitutes more than two
   * orbitals in a spin, with walkers whose reference is nearly singular - and every walker otherwise - on the explicit
   * route (every determinant eliminated on its own); qmc_log_psi and qmc_metropolis keep the excitation tables;
   * qmc_log_derivatives returns the eq. 6 factors with ONE MORE entry, the backflow weight itself (see qmc_n_param);
   * qmc_orbital_derivatives and qmc_nuclear_log_gradient evaluate their AOs at the backflow coordinates (which depend
   * on neither the orbital parameters nor the nuclei); qmc_local_energy_gradient gives the same estimator, not fused
   * (the rows pass through a scratch of the handle); qmc_nuclear_energy_gradient returns QMC_EUNSUPPORTED.  Every
   * Jastrow kernel (D.1, D.2, D.3) combines with backflow: the Jastrow factor and its derivatives sit at r. */
  double backflow_w;
} qmc_system_desc_t;

/* Validate `desc`, preprocess it (shell grouping, excitation tables relative to
 * determinant 0) and upload the constants to `device`.
 * Limits (QMC_EUNSUPPORTED beyond them): n_up, n_dn <= 8; at most 8 distinct
 * virtual (non-reference) orbitals per spin; n_up + n_dn <= 16; n_atoms <= 16;
 * n_ao <= 256; at most 16 distinct orbitals referenced overall.  Determinants that differ
 * from determinant 0 in at most 2 columns per spin take the fast path; more
 * substitutions are evaluated through general k x k sub-determinants (correct, slower).
 * QMC_EINVAL: null pointers, n_up + n_dn == 0, n_det < 1, bad (n,l,m), zeta <= 0,
 * atom / MO index out of range, a determinant list repeating a column.
 * On success *out receives a handle to be released with qmc_destroy. */
int qmc_setup(const qmc_system_desc_t *desc, int device, qmc_system_t **out);

/* Release a handle (device and host memory).  NULL is ignored. */
void qmc_destroy(qmc_system_t *s);

/* Local energy of M walkers (eq. 1-3; trace formulas F.1-F.7, G.7,
 * PAPER.md:290-343, 386).
 *   d_r      device, in : double [n_e][3][M]
 *   d_logpsi device, out: double [M]  log|Psi|                 (may be NULL)
 *   d_sign   device, out: double [M]  sign of Psi: +1, -1 or 0 (may be NULL)
 *   d_eloc   device, out: double [M]  E_L in hartree            (may be NULL)
 * NaN/Inf in the inputs propagate to the outputs.  Asynchronous on cuda_stream. */
int qmc_local_energy(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign,
                     double *d_eloc, void *cuda_stream);

/* qmc_local_energy with HOST buffers (the end-to-end call): h_r host double [n_e][3][M], outputs host
 * double [M] each (any may be NULL).  The walkers are cut into n_chunks contiguous ranges that are
 * pipelined over two internal streams -- strided H2D copy of the range, the kernels, D2H of the three
 * outputs -- so copies overlap computation; page-locked host memory is needed for that overlap, pageable
 * memory works but serialises.  Device scratch (double-buffered, sized for one chunk) belongs to the handle,
 * so concurrent host-variant calls on ONE handle are not allowed.  Synchronous: the outputs are in host
 * memory on return.  Results are identical to qmc_local_energy's (walkers are independent). */
int qmc_local_energy_host(qmc_system_t *s, const double *h_r, int64_t M, double *h_logpsi, double *h_sign,
                          double *h_eloc, int32_t n_chunks);

/* One sampling-and-evaluation step with HOST buffers (what a VMC iteration does between two parameter updates,
 * PAPER.md:180-182): upload the walkers once, n_sweeps Metropolis sweeps (as qmc_metropolis, same random-number
 * stream: the trajectories equal the device call's), E_L of the resulting walkers, batch mean and standard error
 * (eq. 3), walkers and energies back to the host.
 *   h_r host in/out [n_e][3][M];  h_eloc host out [M] (may be NULL);  h_mean, h_stderr host out (may be NULL)
 * The walkers are cut into n_chunks ranges pipelined over the handle's two internal streams (copies of one range
 * overlap the sweeps of the other; page-locked host memory needed for the overlap).  Shares the scratch of
 * qmc_local_energy_host: one host-variant call at a time per handle.  Synchronous. */
int qmc_vmc_step_host(qmc_system_t *s, double *h_r, int64_t M, double step, int32_t n_sweeps, uint64_t seed,
                      uint64_t sweep_offset, int64_t walker_offset, double *h_eloc, double *h_mean, double *h_stderr,
                      int32_t n_chunks);

/* qmc_local_energy with EVERY walker on the explicit route: each determinant's Slater matrices are eliminated on
 * their own (G.7 per determinant; what PAPER.md:349 / Fig. 11 calls "explicit"), no excitation tables.
 * Same arguments, same outputs within rounding; N_det eliminations per walker and spin instead of one.  It exists
 * for the comparison of Fig. 11 (accelerated vs explicit) and as a cross-check; qmc_local_energy uses this route
 * only for walkers whose reference determinant is nearly singular.  Asynchronous. */
int qmc_local_energy_explicit(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign,
                              double *d_eloc, void *cuda_stream);

/* Measurement aid (bench.py's roofline): while enabled, qmc_local_energy / qmc_local_energy_host / qmc_log_derivatives
 * record CUDA events on the stream they launch on -- before the table-path kernel, after it, and after the explicit
 * fallback kernel -- at a cost of three event records per call.  qmc_kernel_times waits for the most recent such call
 * and returns the two device durations in milliseconds (fallback = 0 for a single-determinant system); QMC_EINVAL
 * if timing was never enabled.  One timed call in flight per handle: not for concurrent streams. */
int qmc_set_kernel_timing(qmc_system_t *s, int enabled);
int qmc_kernel_times(qmc_system_t *s, double *h_main_ms, double *h_fallback_ms);

/* log|Psi| and sign only (the part of the path the sampler needs). Same arguments. */
int qmc_log_psi(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign,
                void *cuda_stream);

/* n_sweeps all-electron Metropolis sweeps.  One sweep = one move attempt
 * of every walker: r' = r + step * z, z ~ N(0,1)^(3 n_e); accepted iff
 *   log u < 2 (log|Psi(r')| - log|Psi(r)|),  u uniform on (0,1);
 * a proposal with Psi' = 0 or NaN is rejected.  Random numbers: Philox4x32-10,
 * key = (seed lo32, seed hi32), counter = (w lo32, sweep lo32, j, w hi32) where w is
 * walker_offset + the walker's index in this call and sweep = sweep_offset + s;
 * block j < ceil(3 n_e / 2) gives Box-Muller normals for coordinates 2j, 2j+1
 * (coordinate = 3*electron + xyz), block j = 0xFFFFFFFF gives u.  Two 32-bit words
 * (hi, lo) map to ((hi*2^32 + lo) >> 11 + 1/2) * 2^-53.  Hence a trajectory depends
 * only on (seed, w, sweep), not on batching, and is resumable through sweep_offset.
 *   d_r        device, in/out: double [n_e][3][M]
 *   step       > 0, standard deviation of the proposal per Cartesian coordinate, bohr
 *   d_logpsi   device, out: [M] log|Psi| of the final positions   (may be NULL)
 *   d_sign     device, out: [M]                                    (may be NULL)
 *   d_accept   device, out: uint8 [n_sweeps][M] accept mask        (may be NULL)
 *   d_eloc_acc device, out: [M] sum over the sweeps of E_L evaluated after each sweep
 *              (BASELINE config 5: "E_L on every sweep"); when given, the call alternates
 *              one-sweep sampler launches with the full qmc_local_energy path, so the
 *              energies carry the explicit fallback correction          (may be NULL)
 *   h_n_accepted host, out: total number of accepted moves; if non-NULL the call
 *              synchronises cuda_stream                              (may be NULL)
 * sweep_offset + n_sweeps must be < 2^32. */
int qmc_metropolis(qmc_system_t *s, double *d_r, int64_t M, double step, int32_t n_sweeps, uint64_t seed,
                   uint64_t sweep_offset, int64_t walker_offset, double *d_logpsi, double *d_sign,
                   uint8_t *d_accept, double *d_eloc_acc, int64_t *h_n_accepted, void *cuda_stream);

/* Mean and standard error of the mean of M doubles (eq. 3):
 *   d_x device in [M]; h_mean, h_stderr host out (either may be NULL).
 * Deterministic (fixed reduction tree, compensated).  Synchronises cuda_stream. */
int qmc_batch_stats(const double *d_x, int64_t M, double *h_mean, double *h_stderr, void *cuda_stream);

/* The allocation-free entry point: qmc_batch_stats for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid allocation).  Same reduction, same kernel, but the scratch (block
 * partials and the completion counter) is a fixed file-scope device array of 6400 bytes that every GPU that loads the
 * library holds until the process exits, and the result stays on the device:
 *   d_x   device in  [M], 1 <= M <= 67 108 864 (2^26); a larger M is rejected with QMC_ETOOLARGE
 *   d_out device out [2] = {mean, standard error of the mean}
 * Calls no cudaMalloc / cudaFree / allocating routine; asynchronous on cuda_stream (one 4-byte memset node and one
 * kernel).  qmc_static_scratch_init(device) resolves the array's device address (cudaGetSymbolAddress, once per
 * device); the first qmc_batch_stats_static call on a device does it itself, so call it beforehand when that first call
 * would fall inside a graph capture.  EVERY call on a device shares the one array, which keeps the last call's
 * contents (the call clears what must start at zero): calls that overlap on the GPU -- two streams, or two replays of
 * a captured graph in flight -- race; serialise them.  Deterministic; results equal qmc_batch_stats' up to the
 * rounding order of a different block count. */
int qmc_static_scratch_init(int device);
int qmc_batch_stats_static(const double *d_x, int64_t M, double *d_out, void *cuda_stream);

/* ---- the factors of the gradient estimator, eq. 6 ----
 * Variational parameters handled: theta = (jastrow_a_par, jastrow_a_anti, jastrow_b, jastrow_en_w0,
 * jastrow_en_w1, jastrow_en_w2, then the seven parameters c, a_f, b_f, a_g, b_g, a_h, b_h of every e-e-n term in
 * een_params order (D.3), then d_0 .. d_{n_det-1}); n_param = 6 + 7 n_een + n_det (qmc_n_param).
 * With backflow_w != 0 one more entry follows the CI entries, the backflow weight w of K_BF(r) = w / r:
 *   d ln Psi / d w = sum_n d_n D_n [Tr(A_n^-1 d_w A_n)^up + (..)^dn] / Sigma,  d_w A[i][k] = grad phi_k(rt_i) . sum_{j != i} (r_i - r_j) / r_ij
 * (n_param = 6 + n_det + 1; the Jastrow entries are unchanged, the CI entries are the determinant ratios at the backflow
 * coordinates; from the reference's tables like E_L, the explicit route for walkers with a nearly singular reference).
 * The MO and AO parameters (mu, zeta of PAPER.md:55-57) have their own call, qmc_orbital_derivatives. */
int qmc_n_param(const qmc_system_t *s);

/* qmc_local_energy plus the logarithmic derivatives O_p(r) = (dPsi/dtheta_p)/Psi:
 *   d_O device, out: double [M][n_param] row-major (required)
 * Psi = e^J Sigma (eq. 4): O for a Jastrow parameter is dJ/dtheta from D.1 / D.2 / D.3,
 * O for d_n is D_n^up D_n^dn / Sigma, formed from the excitation tables of the same launch.
 * d_logpsi / d_sign / d_eloc as in qmc_local_energy (E_L carries the explicit fallback
 * correction; O comes from the table path, whose relative error for a nearly singular
 * reference is eps * cond(A_0), not the squared amplification E_L suffers).  Asynchronous. */
int qmc_log_derivatives(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign,
                        double *d_eloc, double *d_O, void *cuda_stream);

/* qmc_local_energy and the estimator of eq. 6 in one pass, the reduction fused into the E_L kernel
 * (SURVEY.md 8(f) NEXT-1): the per-walker derivatives O[w][p] never reach HBM.  Each warp keeps sum_w O_p and
 * sum_w O_p E_L over its walkers in shared memory; groups whose E_L is corrected by the explicit fallback park their
 * rows in a small scratch and are added afterwards with the corrected energies; a final kernel forms
 *   E_v = (1/M) sum_w E_L,   grad_p = (2/M) [ sum_w O_p E_L - (sum_w O_p) E_v ]       (theta as in qmc_n_param)
 * in a fixed order (bit-repeatable).
 *   d_logpsi, d_sign device out [M] (may be NULL);  d_eloc device out [M] (required);
 *   h_Ev host out (may be NULL);  h_grad host out [n_param].
 * Synchronises cuda_stream.  QMC_EUNSUPPORTED when the rows of a warp's walkers do not fit shared memory (very long
 * expansions: use qmc_log_derivatives + qmc_energy_gradient).  For a backflow wavefunction the call runs those two steps
 * itself (n_param includes the backflow weight). */
int qmc_local_energy_gradient(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign, double *d_eloc,
                              double *h_Ev, double *h_grad, void *cuda_stream);

/* Logarithmic derivatives with respect to the orbital parameters:
 *   d_dC    device, out: double [M][n_ao][n_mo]  d ln Psi / d C[beta][alpha] (MO coefficients; the derivative in
 *           the scaling mu_{beta,alpha} of PAPER.md:57 is c_{beta,alpha} times it; zero for MOs no determinant uses)
 *   d_dzeta device, out: double [M][n_ao]        d ln Psi / d zeta_beta, each AO's exponent on its own (with the
 *           standard normalisation d ln N / d zeta = (n + 1/2) / zeta is included; a caller-supplied ao_norm is
 *           taken as independent of zeta)
 * Either may be NULL.  One elimination per spin (the reference's tables); groups of walkers whose reference
 * determinant is nearly singular, (Sigma/D_0)^2 > 1e4, and expansions with more than two substitutions per spin
 * invert every determinant explicitly instead.  Deterministic.  Asynchronous. */
int qmc_orbital_derivatives(qmc_system_t *s, const double *d_r, int64_t M, double *d_dC, double *d_dzeta,
                            void *cuda_stream);

/* Nuclear log-gradient of the wavefunction, grad_alpha ln|Psi| = (1/2) grad_alpha ln rho: the factor of the second
 * term of the force estimator, eq. 7, with the atomic positions as parameters of the AO layer
 * and of the Jastrow kernels that see the nuclei (D.2, D.3):
 *   d_r  device, in:  double [n_e][3][M] walker coordinates (as qmc_local_energy)
 *   d_dR device, out: double [M][n_atoms][3]  d ln|Psi| / d R_alpha,c ; every entry is written
 * d ao_beta(r_i) / d R_alpha = -grad_r ao_beta(r_i) for the AOs of centre alpha, contracted with Gamma = d ln Sigma /
 * d Phi exactly as qmc_orbital_derivatives does (same table path and the same explicit route for near-singular
 * references).  Two launches on cuda_stream (Jastrow part, then the AO part).  Deterministic.  Asynchronous.
 * Returns QMC_EINVAL for null pointers or M <= 0, QMC_EUNSUPPORTED when the shape does not fit shared memory. */
int qmc_nuclear_log_gradient(qmc_system_t *s, const double *d_r, int64_t M, double *d_dR, void *cuda_stream);

/* Nuclear gradient of the local energy, grad_alpha E_L: the first term of the force estimator, eq. 7 (
 * the paper obtains it by automatic differentiation through the AO layer's atomic coordinates; here
 * it is analytic):
 *   d_r  device, in:  double [n_e][3][M]
 *   d_dE device, out: double [M][n_atoms][3]  d E_L / d R_alpha,c ; every entry is written
 * E_L = -1/2 lap Psi / Psi + V of eq. 1-3 with d ao_beta(r_i) / d R_alpha = -grad_r ao_beta(r_i) for the AOs of centre
 * alpha: the AO Hessian and the gradient of the AO Laplacian enter, and d (V_en + V_nn) / d R_alpha (eq. 1).  The
 * chain rule through the determinants collapses into two weight matrices, obtained from the reference's excitation
 * tables (F.6/F.7) by reverse differentiation -- one elimination per spin; groups of walkers whose
 * reference determinant is nearly singular, and expansions with more than two substitutions per spin, eliminate every
 * determinant on its own instead (the explicit route of PAPER.md:349).  Covers the Pade e-e Jastrow D.1 (which does not see the nuclei); with the e-n / e-e-n kernels
 * D.2 / D.3 switched on the call returns QMC_EUNSUPPORTED.  Two launches on cuda_stream.  Deterministic.  Asynchronous.
 * QMC_EINVAL for null pointers or M <= 0. */
int qmc_nuclear_energy_gradient(qmc_system_t *s, const double *d_r, int64_t M, double *d_dE, void *cuda_stream);

/* Force estimator of eq. 7 (reading Q23: the minus sign covers both terms, ln rho = 2 ln|Psi|):
 *   F_alpha = -(1/M) sum_m [ grad_alpha E_L(r_m) + 2 (E_L(r_m) - E_v) grad_alpha ln|Psi(r_m)| ]
 *   d_eloc device in [M]; d_dE (qmc_nuclear_energy_gradient) and d_dlnpsi (qmc_nuclear_log_gradient) device in
 *   [M][n_atoms][3]; h_F host out [n_atoms][3]; h_terms host out [2][n_atoms][3], the two contributions (may be NULL).
 * Deterministic (fixed partition, compensated sums).  Synchronises cuda_stream. */
int qmc_force(const double *d_eloc, const double *d_dE, const double *d_dlnpsi, int64_t M, int32_t n_atoms, double *h_F,
              double *h_terms, void *cuda_stream);

/* Estimator of eq. 6: E_v = mean E_L, grad_p = (2/M) sum_m O[m][p] (E_L[m] - E_v).
 *   d_eloc device in [M]; d_O device in [M][n_param]; h_Ev host out (may be NULL);
 *   h_grad host out [n_param].  Deterministic (fixed partition, compensated sums).
 * Synchronises cuda_stream. */
int qmc_energy_gradient(const double *d_eloc, const double *d_O, int64_t M, int32_t n_param, double *h_Ev,
                        double *h_grad, void *cuda_stream);

/* Measured FP64 throughput of the current device, the roofline denominator of this
 * path (BASELINE.json north_star: "the chip's FP64 peak, measured by a DFMA
 * microbenchmark in the same run").  kind 0: DFMA kernel, 8 independent chains a = fma(a, x, y) per thread; 1: DMMA
 * m8n8k4 kernel; 2: both interleaved in one kernel; probes of the operand forms and of the latency that
 * DESIGN.md section 6 quotes: 3: a = fma(a, x, a), two distinct registers per instruction, 16 chains;
 * 4: a = fma(b, c, a), three distinct registers; 5: ONE dependent chain with one warp per SM sub-partition (the
 * DFMA latency in cycles is 64 n_warps f_clk / rate).  h_tflops host out: best of `reps` launches, counting 2 flops
 * per FMA.  The roofline denominator bench.py uses is the largest of kinds 0, 1 and 3.  Synchronous. */
int qmc_fp64_peak(int device, int kind, int reps, double *h_tflops);

/* Model FP64 work per walker of this system for one E_L evaluation (which = 0) or one
 * Metropolis walker-step (which = 1), in flop-equivalents, by the cost table of
 * DESIGN.md "Roofline" (an FMA counts 2; exp, divide, sqrt, log, sincos by table). */
double qmc_model_flops(const qmc_system_t *s, int which);

/* Number of kernel launches issued by this library on the calling thread since the
 * last call with reset != 0 (bench.py's gpu_launches). */
int64_t qmc_launch_count(int reset);

const char *qmc_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif
