// qmc_device.cuh -- device-side data structures and the warp-synchronous walker
// evaluator of libqmcb200 (sm_100a).  See DESIGN.md "Kernels".
//
// One warp evaluates G = floor(32 / n_e) walkers per pass; lane = g * n_e + e owns
// electron e of walker g in the AO / MO / Jastrow stages, then the warp is re-cut into
// groups of LP lanes, one group per (walker, spin) Gauss-Jordan problem, then into
// groups of LW lanes per walker for the CI sum.  Stages hand over through a per-warp
// shared-memory scratch; only __syncwarp() is used.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qmc {

constexpr int kMaxAtoms = 16;
constexpr int kMaxSpin = 8;   // electrons per spin
constexpr int kMaxVirt = 8;   // distinct virtual orbitals per spin
constexpr int kMaxEen = 6;    // terms of the electron-electron-nucleus Jastrow kernel (D.3; the paper uses 5)
// tuning knobs (defaults are the measured best on B200)
#ifndef QMC_WARPS
#define QMC_WARPS 8          // warps per block
#endif
#ifndef QMC_MINBLOCKS
#define QMC_MINBLOCKS 2      // blocks per SM the register allocation must allow
#endif
#ifndef QMC_MINBLOCKS_EL
#define QMC_MINBLOCKS_EL 2   // ... of the E_L kernels (QMC_WARPS warps per block)
#endif
#ifndef QMC_PAIR_UNROLL
#define QMC_PAIR_UNROLL 2    // unroll factor of the electron-pair loop
#endif
#ifndef QMC_EARLY_INV
#define QMC_EARLY_INV 0      // Gauss-Jordan: invert every pivot candidate before the arg-max is known
#endif
#ifndef QMC_WARPS_PSI
#define QMC_WARPS_PSI 14     // warps per block of the values-only kernels (log|Psi|, Metropolis): 28 warps per SM at 72 registers
                             // (172 bytes of spills) with the compact scratch layout, the most that fits two blocks per SM;
                             // measured per 20 CO sweeps: 10 warps (96 registers, no spills) 5.69 ms, 12 (80 registers) 5.62 /
                             // 5.52 after the record-stream change, 14: 5.39, 16 (one block per SM): 6.46
#endif
#ifndef QMC_WARPS_ORB
#define QMC_WARPS_ORB 10     // warps per block of the orbital-derivative kernel (one block per SM; 8 when shared memory is short; 12 fits but is 40 % slower on bench.py's walkers).
                             // Measured on CO, 32768 walkers, early / equilibrated: 8 warps 0.82 / 0.63 ms, 10: 0.80 / 0.60, 12: 0.78 / 0.80
                             // (12 x 16.3 KB of scratch leave ~30 KB of L1 for the term lists and the constant tables)
#endif
#ifndef QMC_WARPS_PSI_SMALL
#define QMC_WARPS_PSI_SMALL 10  // ... of the instantiations for fewer than 5 electrons per spin (96 registers: 14 warps cost
                                // the Li2 sampler 0.32 -> 0.44 ms per 10 sweeps through the 72-register cap)
#endif
constexpr int kWarpsEl = QMC_WARPS, kWarpsPsi = QMC_WARPS_PSI, kWarpsOrb = QMC_WARPS_ORB, kWarpsOrbSmall = 8;
// launch bound (= most warps per block) of the values-only kernels of an instantiation; qmc_setup launches the
// largest count up to it that still fits two blocks' shared memory on an SM (long expansions: more constants)
template <int NS>
constexpr int kWarpsPsiOf = (NS >= 5) ? QMC_WARPS_PSI : QMC_WARPS_PSI_SMALL;
constexpr int kWarpsBfTab = 8; // warps (= walkers in flight) per block of the backflow E_L kernels: at most this many (fewer
                               // when the per-warp scratch does not fit)
constexpr int kWarpsMax = kWarpsEl > kWarpsPsi ? kWarpsEl : kWarpsPsi;

// shell record kinds
enum : int { SH_S = 0, SH_P = 1, SH_D = 2, SH_P1 = 3, SH_D1 = 4, SH_ATOM = 5, SH_POW = 6 };
// Record stream: per atom {SH_ATOM, the shells with radial power k = 0, then for every further power in use
// {SH_POW k, its shells}}.  SH_POW sets the factor r^k that the hot loop multiplies every following radial function
// by (one multiplication per shell instead of two predicated ones and their selects); the shell records keep k in
// their meta word for the kernels that read them one at a time.
constexpr int kMaxShells = 192;  // shell + atom records; they live in the kernel parameter block (constant bank, uniform data path)

// One shell = the AOs that share a centre, n, l and zeta (one radial factor).  Every lane reads the same
// record, so the records sit in the kernel parameters: the loads go through the uniform data path
// and the constants stay in uniform registers.  48 bytes.
struct ShellRec {
  double zeta;
  double c1;     // 2 zeta (k + l + 1)
  double c2;     // k (k + 2l + 1)
  double kd;     // (double) k,  k = n - 1 - l the radial power
  int32_t meta;  // kind | k << 4 | m << 8 | row in chunk << 12 | flush << 20
  int32_t pad;
  double dlnN;   // d ln(normalisation) / d zeta = (n + 1/2) / zeta, or 0 with a caller-supplied ao_norm (orbital derivatives)
};
// meta fields: kind = SH_*; m = harmonic index of the single-function kinds; row = first AO row of the record
// inside its chunk; flush = 0, or on the last record of a chunk the number of rows the chunk uses
constexpr int kMetaK1 = 1 << 4, kMetaK2 = 2 << 4;

#ifndef QMC_CHUNK
#define QMC_CHUNK 16         // AO rows per DMMA chunk (8 or 16: 2 or 4 k-steps of the m8n8k4 shape)
#endif
constexpr int kChunk = QMC_CHUNK;
// Metropolis: doubles of one sweep's draws per warp: normals [G][3 n_e] (G n_e <= 32), then log u [G]
template <int NS>
constexpr int kDrawDoubles = 96 + ((16 / NS + 1) & ~1);
constexpr int kExpTab = 64;  // entries of the 2^(j/64) table of exp_neg
constexpr int kRngTab = 256; // doubles of the log / sincos tables of the Box-Muller transform

// Constants of the elementary functions (exp_neg, log_pos, sincos_2pi), filled by qmc_setup from the same literal
// expressions the functions used to carry; they travel in the kernel parameter block.
struct MathConsts {
  double e_scale, e_ln2hi, e_ln2lo, e_c5, e_c4, e_c3;            // 64/ln2, -ln2_hi/64, -ln2_lo/64, 1/120, 1/24, 1/6
  double l_c7, l_c6, l_c5, l_c3, l_ln2hi, l_ln2lo;               // 1/7, -1/6, 1/5, 1/3, ln2 hi, ln2 lo
  double s_2pi, s_c7, s_c5, s_c3, s_c8, s_c6, s_c4;              // 2 pi, -1/5040, 1/120, -1/6, 1/40320, -1/720, 1/24
};

// One determinant relative to the reference; the meaning of the two words depends on the class (qmc_setup):
// one or two byte offsets of table entries (class 1, 2), four 16-bit byte offsets {11,12 | 21,22} of a 2x2
// block (class 3), or per spin four 8-bit entry indices {11,12,21,22} where unused slots point at the
// constant entries TS-2 (= 1.0 in T, 0 in M) and TS-1 (= 0.0) (class 4).  16 bytes.
struct __align__(16) DetRec {
  uint32_t up, dn;  // 4 x uint8 each
  double d;
};

// A determinant with more than two substitutions in one spin (rare; general k x k sub-determinants).
struct GenSpin {
  uint8_t k;
  uint8_t p[kMaxSpin];  // substituted reference positions
  uint8_t q[kMaxSpin];  // virtual indices
  uint8_t pad[7];
};
struct GenDet {  // 56 bytes
  double d;
  GenSpin s[2];
};

// Column lists of every determinant (caller order), for the explicit fallback path.  24 bytes.
struct DetCols {
  int8_t col[2][kMaxSpin];  // kernel MO column of position j, per spin
  double d;
};

// A walker is re-evaluated with every determinant eliminated explicitly when (Sigma / D_0)^2 exceeds
// kFallbackK max(1, |E_L|): the table path (F.6/F.7) loses about log10((Sigma/D_0)^2) digits when the
// reference determinant is nearly singular while the expansion is not.  Measured:
// E_L error ~ 1.2e-15 (Sigma/D_0)^2, so K = 8e5 keeps it below 1e-9 max(1, |E_L|), a tenth of the parity bound.
#ifndef QMC_FALLBACK_K
#define QMC_FALLBACK_K 8.0e5
#endif
constexpr double kFallbackK = QMC_FALLBACK_K;
// ... and in any case when |Sigma / D_0| > 1e4: log|Psi| of the table path is off by ~1e-15 |Sigma/D_0| (1e-12 at
// 1024), and its parity bound 1e-10 is ABSOLUTE, so walkers with a huge |E_L| must not escape through the first test.
#ifndef QMC_FALLBACK_CAP
#define QMC_FALLBACK_CAP 1.0e8
#endif
constexpr double kFallbackCap = QMC_FALLBACK_CAP;
// The same loss when the reference ALONE is nearly singular while Sigma / D_0 stays moderate (the CI coefficients of
// the large determinants are small): T, G, H carry relative errors eps * cond(A_0) and their O(cond^2) parts cancel.
// kappa = max |T[p][q]| of a spin estimates cond(A_0) at no cost.  Measured on all 131072 CO, 32768 Li2 and
// 32768 CO-500 walkers against the oracle (its long-double build) with the fallback off: worst error of
// a walker with kappa^2 <= 1e6 max(1, |E_L|) is 2.8e-10 max(1, |E_L|); 0.12% / 0.16% / 0.07% of the walkers exceed it.
// (The (Sigma/D_0)^2 test alone left a CO walker at 2.0e-7: kappa 4.8e4, Sigma/D_0 = -118.)
#ifndef QMC_FALLBACK_KAPPA
#define QMC_FALLBACK_KAPPA 1.0e6
#endif
constexpr double kFallbackKappa = QMC_FALLBACK_KAPPA;
constexpr double kFallbackKappaCap = (QMC_FALLBACK_KAPPA > 1.0e100) ? QMC_FALLBACK_KAPPA : 1.0e10;
// Orbital-parameter derivatives: the table-path error of Gamma is ~1.2e-15 (Sigma/D_0)^2 of the walker's largest
// derivative (measured); beyond (Sigma/D_0)^2 = 1e4 the group takes the explicit route.
#ifndef QMC_FALLBACK_ORB
#define QMC_FALLBACK_ORB 1.0e4
#endif
#ifndef QMC_FALLBACK_ORB_KAPPA
#define QMC_FALLBACK_ORB_KAPPA 1.0e6
#endif
constexpr double kFallbackOrb = QMC_FALLBACK_ORB;
constexpr double kFallbackOrbKappa = QMC_FALLBACK_ORB_KAPPA;  // ... or kappa^2 beyond 1e6 (same conditioning estimate as E_L's)

// One term of Y[spin][p][q] = d(Sigma/D_0)/dT[p][q]: w * R_other * T_spin[cof]  (w = d_n times the cofactor's sign;
// oth = the other spin's 2x2 code {i11, i12, i21, i22} as in class-4 DetRec, constant slots for k < 2;
// cof = table index of the cofactor entry, the constant-1 slot for a single substitution)
struct __align__(16) YRec {
  double w;
  uint32_t oth;
  uint16_t cof, pad;
};

struct SysParams {  // passed by value to every kernel
  MathConsts mc;
  int n_atoms, n_up, n_dn, n_e;
  int n_shell, n_ao, n_mo, n_det;  // n_shell = records of the shell/atom stream; n_mo = orbitals referenced (kernel
                                   // order); n_det = packed determinant records (classes 1-4)
  int n_a1, n_a2, n_b;             // class boundaries in dets[]: [0,n_a1) one entry, [n_a1,n_a2) two entries,
                                   // [n_a2,n_b) one 2x2 block, [n_b,n_det) two 2x2 blocks (qmc_setup)
  double d_ref;                    // summed coefficients of the determinants equal to the reference
  int n_ref;                       // how many determinants equal the reference
  const int *det_orig;             // device [n_det_all]: caller's index of the determinants in kernel order
  const YRec *yrec;                // device: gather lists of Y = d(Sigma/D_0)/dT, one list per table entry
  const int2 *ytgt;                // device [n_ytgt + 1]: {entry index in the walker's (up, down) tables, list start}
  int n_ytgt;
                                   // (reference-equal ones, then dets[] classes 1-4, then gen[])
  int nv[2];                       // virtual orbitals per spin
  int G;                           // walkers per warp pass
  int smem_const_bytes;
  int c_doubles;                   // size of the C fragment table
  int n_chunks;                    // AO chunks of kChunk rows
  double a_par, a_anti, b, vnn;
  double bf_w;                     // inverse backflow kernel K_BF(r) = bf_w / r; 0 = none
  double en_w0, en_w1, en_w2;      // electron-nucleus Jastrow kernel (D.2); has_en = 0 when w0 = w1 = 0
  int has_en;
  int n_een;                       // electron-electron-nucleus kernel (D.3): terms (c, a1, b1, a2, b2, a3, b3)
  double een[kMaxEen][7];
  double atom[kMaxAtoms][4];       // x, y, z, Z
  int8_t ref_col[2][kMaxSpin];     // kernel MO column of reference position j, per spin
  int8_t virt_col[2][kMaxVirt];    // kernel MO column of virtual q, per spin
  ShellRec shells[kMaxShells];     // [n_shell] record stream: {SH_ATOM a, shells of a} per atom (n_shell counts both)
  const double *exp_tab;           // device [kExpTab]: 2^(j/64), correctly rounded (qmc_setup)
  const double *rng_tab;           // device [kRngTab]: log and sincos tables of the Box-Muller transform
  const double *C;                 // device [chunk][k-step 4][MO tile NT][lane 32]: DMMA B fragments of
                                   // N_ao * C (normalisation folded in, zero padded), see qmc_setup
  const DetRec *dets;              // device [n_det]  (at most two substitutions per spin)
  const GenDet *gen;               // device [n_gen]  (the others)
  int n_gen;
  int n_det_all;                   // all determinants
  const DetCols *det_cols;         // device [n_det_all]
  // orbital-parameter derivatives (qmc_orbital_derivatives): kernel AO row -> caller's AO index (-1 = padding row)
  // and normalisation, kernel MO column -> caller's MO index
  const int *ao_orig;              // device [n_chunks * kChunk]
  const double *ao_nrm;            // device [n_chunks * kChunk]
  int mo_orig[16];
  int n_mo_all;                    // MOs of the caller's coefficient matrix
};

struct WalkerIO {
  // explicit-fallback work list: groups whose walkers need re-evaluation (filled by the fast kernel)
  int *fb_list;        // device [ceil(M / G)] group indices, or null
  int *fb_count;       // device counter
  int *fb_done;        // device [ceil(M / G)] per listed group: slices finished (zeroed when the group is listed)
  double *fb_part;     // device [items][G][2] partial sums {Sigma, Sum d D t} of the explicit kernel's work items
  const double *r_in;  // [n_e][3][M]
  double *r_out;       // Metropolis: same buffer
  double *logpsi, *sign, *eloc;
  double *O;           // device [M][kJastrowParams + 7 n_een + n_det_all] parameter derivatives (DerivOut), or null
  int64_t M;
  // fused eq. 6 reduction (qmc_local_energy_gradient): per-warp partial sums and the O rows of the listed groups
  double *fuse_part;   // device [2 n_param + 1][grid warps]: sum O_p, sum O_p E_L, then sum E_L
  double *fb_O;        // device [fb_cap][G][n_param]: O rows of the groups on the explicit work list
  int fb_cap;          // rows of fb_O; a listed group beyond it sets fb_over
  int *fb_over;        // device flag
  int fuse_stride;     // doubles each warp's scratch is extended by: (G + 2) n_param, even
};

// Parameter-derivative output (eq. 6): O[w][p] = (dPsi/dtheta_p)/Psi for
// theta = (a_par, a_anti, b, en_w0, en_w1, en_w2, {c, a_f, b_f, a_g, b_g, a_h, b_h} of every e-e-n term,
// d_0 .. d_{n_det-1}); row-major [M][kJastrowParams + 7 n_een + n_det_all].
constexpr int kJastrowParams = 6;
struct DerivOut {
  double *O;      // device, or null
  int64_t w0;     // first walker of the group being evaluated
  int64_t M;
};

struct MetroParams {
  double step;
  int n_sweeps;
  uint32_t key0, key1;
  uint32_t sweep0;
  int64_t walker_offset;
  uint8_t *accept;       // [n_sweeps][M] or null
  int resume;            // 1: log|Psi| and sign of the starting positions are in io.logpsi / io.sign (as a
                         // previous launch left them) instead of being evaluated
  unsigned long long *n_accepted;  // device counter or null
};

__host__ __device__ constexpr int pow2ceil(int x) {
  int p = 1;
  while (p < x) p <<= 1;
  return p;
}
__host__ __device__ constexpr int pow2floor(int x) {
  int p = 1;
  while (2 * p <= x) p <<= 1;
  return p;
}
__host__ __device__ constexpr int cmax(int a, int b) { return a > b ? a : b; }

// compile-time geometry of one instantiation
template <int NS, int NMO>
struct Geo {
  static constexpr int NV = (NMO - NS) > 0 ? ((NMO - NS) < kMaxVirt ? (NMO - NS) : kMaxVirt) : 0;
  static constexpr int LP = pow2ceil(cmax(cmax(NS, NV), 1));  // lanes per Gauss-Jordan problem
  static constexpr int PP = 32 / LP;                          // problems per pass
  static constexpr int GMAX = 16 / NS;                        // walkers per warp pass (host: G <= GMAX)
  static constexpr int ROWS = (2 * GMAX * NS) < 32 ? (2 * GMAX * NS) : 32;  // electron rows of a pass
  static constexpr int RS = LP + 1;       // table row stride: odd, so that the entries (p, q) of one virtual q and
                                          // different positions p fall into different banks (CI-sum lookups)
  static constexpr int TS = NS * RS + 2;  // table stride per problem: T[p][q] entries + {1.0, 0.0}
  __host__ __device__ static constexpr int even(int x) { return (x + 1) & ~1; }
  // per-warp scratch, in doubles (all offsets even: 16-byte aligned).
  // When one Gauss-Jordan pass covers all 2 GMAX problems (SINGLE), the MO rows are in registers
  // before the first table entry is written, so G, T and M reuse the space of Phi and B.
  // MO rows (Phi, B).  In the E_L kernels with two 8-column tiles the row stride is 16 and odd rows swap their
  // two halves (column ^ 8): the D-fragment stores of the contraction (two adjacent rows per quarter-warp)
  // and the Gauss-Jordan loads (rows of two problems per half-warp, 7 rows apart) then hit disjoint banks
  // (measured: E_L kernel -1.3%; the values-only kernels lose more to the index arithmetic than they gain).
  static constexpr int NTc = (NMO + 7) / 8;
  static constexpr bool SWZ = NTc == 2;
  __host__ __device__ static constexpr int moIdx(bool el, int row, int col) {
    return (SWZ && el) ? row * 16 + (col ^ ((row & 1) << 3)) : row * NMO + col;
  }
  static constexpr int szPhi = even(ROWS * (SWZ ? 16 : NMO));
  static constexpr int szG = even(cmax(PP * NS * NS, 2));
  static constexpr int szT = even(cmax(2 * GMAX * TS, 96 + 32));
  static constexpr int szM = even(2 * GMAX * TS);
  static constexpr bool SINGLE = (2 * GMAX <= PP) && (2 * szPhi >= szG + szT + szM);
  static constexpr int oPhi = 0;
  static constexpr int oB = oPhi + szPhi;
  static constexpr int oG = SINGLE ? 0 : oB + szPhi;
  static constexpr int oT = oG + szG;
  static constexpr int oM = oT + szT;
  static constexpr int oPart = SINGLE ? oB + szPhi : oM + szM;
  static constexpr int oXYZ = oPart + 64;                     // coordinates (pair loop)
  static constexpr int oProb = oXYZ + 96;
  static constexpr int oRes = oProb + 2 * GMAX * 4;           // per walker {log|Psi|, sign, E_L, -}
  static constexpr int layout_total = oRes + GMAX * 4;
  // Compact layout of the values-only evaluator (log|Psi| kernel, sampler): no operator rows B, no G staging, no M
  // tables -- the per-electron scalars, coordinates and results follow the values-only AO tile / the T tables
  // directly (CO: 760 doubles per warp instead of 1088), which is what lets 24 warps share an SM.
  static constexpr int psiBase = even(cmax(cmax(kChunk * 36, oT + szT), szPhi));
  __host__ __device__ static constexpr int oPartC(bool c) { return c ? psiBase : oPart; }
  __host__ __device__ static constexpr int oXYZC(bool c) { return oPartC(c) + 64; }
  __host__ __device__ static constexpr int oProbC(bool c) { return oXYZC(c) + 96; }
  __host__ __device__ static constexpr int oResC(bool c) { return oProbC(c) + 2 * GMAX * 4; }
  // DMMA contraction scratch, from offset 0 (everything it overlays is dead while it is live): the AO
  // tile [kChunk AO rows][S].  Column = lane for the AO values; for E_L the combined operator of the
  // lane sits in column opCol(lane) >= 32, so every lane (also one that owns no electron) stores
  // unconditionally.  The m8n8k4 A fragments read 8 columns per M-tile: VT full tiles of values, then --
  // when ROWS = 8 VT + 4 -- one MERGED tile {4 value columns, 4 operator columns}, then the operator
  // tiles.  S = 4 (mod 16): a half-warp of a fragment load (4 k-rows x 4 columns of doubles) then covers
  // all 32 banks once (measured with S = 8 (mod 16): 2-way conflicts, 4 wavefronts per load instead of 2).
  static constexpr int S1 = 36, S2 = 68;                      // tile row stride: values only / with operator
  static constexpr int VT = ROWS / 8;                         // full value tiles
  static constexpr bool MERGE = (ROWS % 8) == 4;
  static constexpr int VTc = (ROWS + 7) / 8;
  __host__ __device__ static constexpr int mTiles(bool el) { return el ? (MERGE ? 2 * VT + 1 : 2 * VTc) : VTc; }
  // operator column of a lane: 32 + lane; behind the merged tile the real rows move up by 4 (columns
  // 60..63 for ROWS = 28) and the lanes that own no row park in the free columns 56..59, which no fragment
  // reads and whose banks no other lane of their half-warp touches
  __host__ __device__ static constexpr int opCol(int lane) {
    return !MERGE ? 32 + lane : (lane < 8 * VT ? 32 + lane : (lane < ROWS ? 36 + lane : 28 + lane));
  }
  // first tile column of M-tile m minus the fragment row (the merged tile adds mergeShift(fr))
  __host__ __device__ static constexpr int tileCol(bool el, int m) {
    return !el ? 8 * m : (MERGE ? (m <= VT ? 8 * m : 32 + 8 * (m - VT - 1)) : (m < VTc ? 8 * m : 32 + 8 * (m - VTc)));
  }
  __host__ __device__ static constexpr int mergeShift(int fr) { return (fr & 4) << 3; }  // rows 4..7: + 32
  static constexpr int total = cmax(layout_total, kChunk * S2);
  __host__ __device__ static constexpr int totalC(bool c) { return c ? oResC(true) + GMAX * 4 : total; }
  static constexpr int NT = (NMO + 7) / 8;                    // 8-column MO tiles
  // orbital-derivative kernel only: behind the common scratch, Gamma [ROWS][NMO], then the inverses of one determinant's
  // problems [2 GMAX][NS][NS] and their column indices [2 GMAX][NS] (ints)
  static constexpr int oGam = total;
  static constexpr int oInv = oGam + even(ROWS * NMO);
  static constexpr int oCol = oInv + even(2 * GMAX * NS * NS);
  static constexpr int oY = oCol + even(GMAX * NS);        // table path: Y = d den / d T, laid out like the T tables
  static constexpr int orbExtra = even(ROWS * NMO) + even(2 * GMAX * NS * NS) + even(GMAX * NS) + even(2 * GMAX * TS);
  // nuclear energy-gradient kernel only (eval_walkers<..., ORB = 3>), behind the orbital-derivative extras: the second
  // weight matrix Gamma2 [ROWS][NMO], grad_i J [3][32], the staging of A_n^-1 B_n for one pass of problems
  // [PP][NS][NS] and X_n = A_n^-1 B_n A_n^-1 of one determinant's problems [2 GMAX][NS][NS]
  static constexpr int oGam2 = oY + even(2 * GMAX * TS);
  static constexpr int oGJ = oGam2 + even(ROWS * NMO);
  static constexpr int oStage = oGJ + 96;
  static constexpr int oX = oStage + even(PP * NS * NS);
  // ... and for its table route (ORB = 4): H = A0^-1 Bv [2 GMAX][NS][LP] and Z = d num / d T, laid out like the T tables
  static constexpr int oH = oX + even(2 * GMAX * NS * NS);
  static constexpr int oZ = oH + even(2 * GMAX * NS * LP);
  static constexpr int frcExtra = orbExtra + even(ROWS * NMO) + 96 + even(PP * NS * NS) + even(2 * GMAX * NS * NS) +
                                  even(2 * GMAX * NS * LP) + even(2 * GMAX * TS);
  static_assert(oZ + even(2 * GMAX * TS) == total + frcExtra, "force-kernel scratch regions do not add up");
  // bounds of the overlays (compile-time hygiene: no memory checker runs on this pool)
  static_assert(NS >= 1 && NS <= kMaxSpin && NMO <= 16, "instantiation outside the register-array limits");
  static_assert(ROWS <= 32 && 2 * GMAX * NS >= ROWS, "electron rows of a pass exceed the warp");
  static_assert(opCol(31) < S2 && 31 < S1, "tile columns exceed the row stride");
  static_assert(tileCol(true, mTiles(true) - 1) + 7 < S2 && (!MERGE || tileCol(true, VT) + 7 + mergeShift(7) < S2),
                "operator tiles exceed the row stride");
  static_assert(kChunk * S2 <= total && layout_total <= total, "scratch smaller than its overlays");
  static_assert(oB + szPhi <= oPart, "MO rows overlap the per-electron scalars");
  static_assert(SINGLE ? (oM + szM <= oPart) : true, "tables overlap the per-electron scalars");
  static_assert(2 * GMAX * TS * 2 <= szT + szM, "interleaved {T, M} tables exceed their region");
  static_assert(NS * RS + 1 < 256 && 8 * (2 * TS) < 65536, "table indices exceed the packed determinant records");
};

// ---------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al.), counter-based; reading Q9
// ---------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int i = 0; i < 10; ++i) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__device__ __forceinline__ double u53(uint32_t hi, uint32_t lo) {
  unsigned long long v = (((unsigned long long)hi << 32) | lo) >> 11;
  return ((double)v + 0.5) * (1.0 / 9007199254740992.0);
}

// Fast FP64 reciprocal / reciprocal square root: MUFU seed (about 20 bits) + two Newton steps
// (relative error ~1e-16; inputs here are distances and pivots, never subnormal).
__device__ __forceinline__ double rcp_fast(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  y = fma(y, e, y);
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
}
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double h = 0.5 * x;
  double e = fma(-h * y, y, 0.5);
  y = fma(y, e, y);
  e = fma(-h * y, y, 0.5);
  return fma(y, e, y);
}

// exp(x) for x <= 0 (STO radial factors e^{-zeta r}): x = (64 n + j) ln2/64 + f, |f| <= ln2/128,
//   e^x = 2^n * 2^(j/64) * (1 + q(f)),  q = f + f^2 (1/2 + f/6 + f^2 (1/24 + f/120))   (truncation 3.5e-17)
// with 2^(j/64) from a 64-entry shared-memory table (correctly rounded doubles, built by qmc_setup) and
// 2^n applied to the exponent field.  Arguments below -690 are clamped (value ~1e-300, zero for every
// use here) by one unsigned minimum on the high word (negative doubles order like their bit patterns); the clamp
// also swallows a NaN argument -- a NaN coordinate still reaches log|Psi| and E_L through the distances of
// the Jastrow factor and the potential.
// The constants come from the kernel parameter block (MathConsts): an FP64 instruction takes one of them straight
// from the constant bank; as literals each cost two 32-bit moves per use (measured: 12 of the 33 instructions).
__device__ __forceinline__ double exp_neg(double x, const double *__restrict__ tab, const MathConsts &K) {
  constexpr double kMagic = 6755399441055744.0;  // 1.5 * 2^52
  x = __hiloint2double((int)min((unsigned)__double2hiint(x), 0xC0859000u), __double2loint(x));  // x >= -690
  const double t = fma(x, K.e_scale, kMagic);  // round(64 x / ln2) in the low mantissa bits
  const int n = __double2loint(t);
  const double nd = t - kMagic;
  double f = fma(nd, K.e_ln2hi, x);
  f = fma(nd, K.e_ln2lo, f);
  const double f2 = f * f;
  const double a = fma(f, K.e_c5, K.e_c4), b = fma(f, K.e_c3, 0.5);
  const double q = fma(f2, fma(f2, a, b), f);
  const double T = tab[n & (kExpTab - 1)];
  const double p = fma(T, q, T);
  return __hiloint2double(__double2hiint(p) + ((n >> 6) << 20), __double2loint(p));
}

// The same with the table given as a 32-bit shared-memory address held in a register (the hot AO loop: the generic
// pointer made the compiler rebuild the shared window base -- S2UR + two ULEA -- at every call).
__device__ __forceinline__ double exp_neg_s32(double x, uint32_t tab32, const MathConsts &K) {
  constexpr double kMagic = 6755399441055744.0;
  x = __hiloint2double((int)min((unsigned)__double2hiint(x), 0xC0859000u), __double2loint(x));
  const double t = fma(x, K.e_scale, kMagic);
  const int n = __double2loint(t);
  const double nd = t - kMagic;
  double f = fma(nd, K.e_ln2hi, x);
  f = fma(nd, K.e_ln2lo, f);
  const double f2 = f * f;
  const double a = fma(f, K.e_c5, K.e_c4), b = fma(f, K.e_c3, 0.5);
  const double q = fma(f2, fma(f2, a, b), f);
  double T;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(T) : "r"(tab32 + (uint32_t)((n & (kExpTab - 1)) << 3)));
  const double p = fma(T, q, T);
  return __hiloint2double(__double2hiint(p) + ((n >> 6) << 20), __double2loint(p));
}

// ---------------------------------------------------------------------------------
// Elementary functions of the Box-Muller transform (reading Q9), table-driven so that one
// normal pair costs ~40 FP64 instructions.  Tables are built in long double by qmc_setup (kRngTab
// doubles: 64 {1/c_j, -log(1/c_j)} pairs, then 64 {cos, sin}(2 pi j / 64) pairs) and sit in shared memory.
// ---------------------------------------------------------------------------------
// log(u) for a positive normal u: u = 2^e m, m in [sqrt(1/2), sqrt(2)); the top six bits
// of m's offset in that range select c_j; r = m / c_j - 1, |r| <= 0.0079;
// log u = e ln2 - log(1/c_j) + (r - r^2/2 + ... + r^7/7)      (truncation r^8/8 < 2e-18)
__device__ __forceinline__ double log_pos(double u, const double2 *__restrict__ tab, const MathConsts &K) {
  int hx = __double2hiint(u) + (0x3ff00000 - 0x3fe6a09e);
  const int e = (hx >> 20) - 1023;
  hx &= 0xfffff;
  const double m = __hiloint2double(hx + 0x3fe6a09e, __double2loint(u));
  const double2 t = tab[hx >> 14];
  const double r = fma(m, t.x, -1.0);
  double p = fma(r, K.l_c7, K.l_c6);
  p = fma(p, r, K.l_c5);
  p = fma(p, r, -0.25);
  p = fma(p, r, K.l_c3);
  p = fma(p, r, -0.5);
  const double lg = fma(r * r, p, r);
  const double ed = (double)e;
  return fma(ed, K.l_ln2hi, t.y) + fma(ed, K.l_ln2lo, lg);  // ln2 hi, lo
}
// sqrt(x), x > 0 normal: x * rsqrt(x) with one correction step (error < 1 ulp)
__device__ __forceinline__ double sqrt_pos(double x) {
  const double y = rsqrt_fast(x);
  const double s = x * y;
  return fma(fma(-s, s, x), 0.5 * y, s);
}
// sin and cos of 2 pi u, u in [0,1): u = j/64 + f, |f| <= 1/128 (exact), a = 2 pi f, |a| <= 0.0491;
// short Taylor polynomials in a (truncation < 5e-18) rotated by the tabulated {cos, sin}(2 pi j/64).
__device__ __forceinline__ void sincos_2pi(double u, const double2 *__restrict__ tab, const MathConsts &K, double &sn, double &cs) {
  constexpr double kMagic = 6755399441055744.0;  // 1.5 * 2^52
  const double t = fma(u, 64.0, kMagic);  // round(64 u) in the low mantissa bits
  const double f = fma(t - kMagic, -1.0 / 64, u);
  const double2 w = tab[__double2loint(t) & 63];
  const double a = f * K.s_2pi;
  const double a2 = a * a;
  const double sa = fma(a * a2, fma(a2, fma(a2, K.s_c7, K.s_c5), K.s_c3), a);                 // sin a
  const double qc = a2 * fma(a2, fma(a2, fma(a2, K.s_c8, K.s_c6), K.s_c4), -0.5);             // cos a - 1
  cs = fma(-w.y, sa, fma(w.x, qc, w.x));
  sn = fma(w.x, sa, fma(w.y, qc, w.y));
}

// FP64 tensor-core MMA, D(8x8) += A(8x4) B(4x8).  Fragments (lane = 4 r + k):
//   A[r][k] in lane 4r+k;  B[k][n] in lane 4n+k;  D[r][2k], D[r][2k+1] in lane 4r+k.
__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

// Shared-memory stores through an explicit 32-bit shared address that the compiler cannot rematerialise
// (opaque_u32): keeps one address register live instead of recomputing lane offsets at every store.
__device__ __forceinline__ uint32_t opaque_u32(uint32_t v) {
  asm volatile("" : "+r"(v));
  return v;
}
template <int BYTE_OFF>
__device__ __forceinline__ void sts_f64(uint32_t addr, double v) {
  asm volatile("st.shared.f64 [%0+%1], %2;" ::"r"(addr), "n"(BYTE_OFF), "d"(v) : "memory");
}

__device__ __forceinline__ double shfl_d(double v, int src, int width) {
  return __shfl_sync(0xffffffffu, v, src, width);
}
__device__ __forceinline__ double shfl_xor_d(double v, int mask) { return __shfl_xor_sync(0xffffffffu, v, mask); }

}  // namespace qmc
