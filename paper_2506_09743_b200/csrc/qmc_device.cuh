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
constexpr int kWarpsPerBlock = 4;

// shell record kinds
enum : int { SH_S = 0, SH_P = 1, SH_D = 2, SH_P1 = 3, SH_D1 = 4 };

struct ShellRec {  // 32 bytes
  double zeta;
  double c1;     // 2 zeta (k + l + 1)
  float c2;      // k (k + 2l + 1)
  int16_t kind;  // SH_*
  int16_t k;     // radial power n-1-l
  int16_t m;     // harmonic index for the single-function kinds
  int16_t ao0;   // first AO row (kernel order) of this record
  int32_t pad;
};

struct DetRec {  // 16 bytes.  exc: bits 0-3 k, 4-7 p1, 8-11 q1, 12-15 p2, 16-19 q2
  uint32_t up, dn;
  double d;
};

struct SysParams {  // passed by value to every kernel
  int n_atoms, n_up, n_dn, n_e;
  int n_shell, n_ao, n_mo, n_det;  // n_mo = orbitals referenced (kernel order)
  int nv[2];                       // virtual orbitals per spin
  int G;                           // walkers per warp pass
  int smem_const_bytes;
  double a_par, a_anti, b, vnn;
  double atom[kMaxAtoms][4];       // x, y, z, Z
  int shell_begin[kMaxAtoms + 1];  // shells of atom a: [shell_begin[a], shell_begin[a+1])
  int8_t ref_col[2][kMaxSpin];     // kernel MO column of reference position j, per spin
  int8_t virt_col[2][kMaxVirt];    // kernel MO column of virtual q, per spin
  const ShellRec *shells;          // device [n_shell]
  const double *C;                 // device [n_ao][NMO]  (normalisation folded in, zero padded)
  const DetRec *dets;              // device [n_det]
};

struct WalkerIO {
  const double *r_in;  // [n_e][3][M]
  double *r_out;       // Metropolis: same buffer
  double *logpsi, *sign, *eloc;
  int64_t M;
};

struct MetroParams {
  double step;
  int n_sweeps;
  uint32_t key0, key1;
  uint32_t sweep0;
  int64_t walker_offset;
  uint8_t *accept;       // [n_sweeps][M] or null
  double *eloc_acc;      // [M] or null
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
  // per-warp scratch, in doubles
  static constexpr int oPhi = 0;
  static constexpr int oB = oPhi + 32 * NMO;
  static constexpr int oXYZ = oB + 32 * NMO;
  static constexpr int oPart = oXYZ + 96;
  static constexpr int oG = oPart + 64;
  static constexpr int oT = oG + PP * NS * NS;
  static constexpr int oM = oT + 32 * LP;   // 2G*NS <= 32 rows of LP entries
  static constexpr int oProb = oM + 32 * LP;
  static constexpr int oProp = oProb + 32 * 4;  // Metropolis: proposals z [G][3 n_e] + log u [G]
  static constexpr int oRes = oProp + 96 + 32;   // per walker {log|Psi|, sign, E_L}
  static constexpr int total = oRes + 96;
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

__device__ __forceinline__ double shfl_d(double v, int src, int width) {
  return __shfl_sync(0xffffffffu, v, src, width);
}
__device__ __forceinline__ double shfl_xor_d(double v, int mask) { return __shfl_xor_sync(0xffffffffu, v, mask); }

}  // namespace qmc
