// qmc_kernels.cuh -- __global__ entry points: local energy / log psi, persistent
// Metropolis, batch statistics.  One warp = G walkers per pass, grid-stride over groups.
#pragma once
#include "qmc_eval.cuh"
#include "qmc_backflow.cuh"

namespace qmc {

// copy the constants into shared memory; returns pointers.  Layout: C | exp table | rng tables | dets.
template <int NMO>
__device__ __forceinline__ void load_constants(const SysParams &P, unsigned char *smem, const double *&sC,
                                               const double *&sExp, const DetRec *&sDet, double *&wsBase) {
  double *c = reinterpret_cast<double *>(smem);
  const int nC = P.c_doubles;
  for (int i = threadIdx.x; i < nC; i += blockDim.x) c[i] = P.C[i];
  double *et = c + nC;
  for (int i = threadIdx.x; i < kExpTab; i += blockDim.x) et[i] = P.exp_tab[i];
  for (int i = threadIdx.x; i < kRngTab; i += blockDim.x) et[kExpTab + i] = P.rng_tab[i];
  DetRec *dt = reinterpret_cast<DetRec *>(et + kExpTab + kRngTab);
  {
    const double *src = reinterpret_cast<const double *>(P.dets);
    double *dst = reinterpret_cast<double *>(dt);
    for (int i = threadIdx.x; i < P.n_det * 2; i += blockDim.x) dst[i] = src[i];
  }
  sC = c;
  sExp = et;
  sDet = dt;
  wsBase = reinterpret_cast<double *>(smem + P.smem_const_bytes);
  __syncthreads();
}

// benign coordinates for lanes that own no electron (results are discarded)
__device__ __forceinline__ void dummy_xyz(int lane, double &x, double &y, double &z) {
  x = 0.37 + 0.11 * lane;
  y = -0.21 + 0.07 * lane;
  z = 0.53 - 0.05 * lane;
}

// FUSE (with DERIV): the eq. 6 reduction is fused: the rows O[w][:] stay in shared memory,
// each warp keeps sum_w O_p and sum_w O_p E_L over its walkers and writes them once at the end; a group on the explicit
// work list (its E_L is corrected later) parks its rows in io.fb_O instead; fused_gradient_final_kernel finishes.
template <int NS, int NMO, bool EL, bool X, int WPB, bool DERIV = false, bool EEN = false, bool BF = false, bool FUSE = false>
__global__ void __launch_bounds__(WPB * 32, EL ? QMC_MINBLOCKS_EL : QMC_MINBLOCKS)
    local_energy_kernel(const __grid_constant__ SysParams P, const WalkerIO io) {
  extern __shared__ __align__(16) unsigned char smem[];
  const double *sC;
  const double *sExp;
  const DetRec *sDet;
  double *wsBase;
  load_constants<NMO>(P, smem, sC, sExp, sDet, wsBase);
  using GE = Geo<NS, NMO>;
  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;  // shfl: tells the compiler it is warp-uniform
  constexpr bool CP = kCompact<EL, false, 0>;
  double *ws = wsBase + warp * (GE::totalC(CP) + (FUSE ? io.fuse_stride : 0));
  const int ne = X ? 2 * NS : P.n_e, G = X ? GE::GMAX : P.G;
  const int g = lane / ne, e = lane - g * ne;
  const int64_t n_groups = (io.M + G - 1) / G;
  const int wpb = (int)(blockDim.x >> 5);  // warps launched per block (<= WPB, the launch bound)
  const int64_t stride = (int64_t)gridDim.x * wpb;
  const int np = kJastrowParams + 7 * P.n_een + P.n_det_all;
  double *sO = ws + GE::total, *accO = sO + G * np, *accOE = accO + np;  // FUSE only
  double accE = 0.0;
  if (FUSE) {
    for (int p = lane; p < 2 * np; p += 32) accO[p] = 0.0;
    __syncwarp();
  }
  auto fetch = [&](int64_t grp, double &x, double &y, double &z) {
    const int64_t w = grp * G + g;
    if ((g < G) && (w < io.M)) {
      x = __ldg(io.r_in + ((int64_t)e * 3 + 0) * io.M + w);
      y = __ldg(io.r_in + ((int64_t)e * 3 + 1) * io.M + w);
      z = __ldg(io.r_in + ((int64_t)e * 3 + 2) * io.M + w);
    } else {
      dummy_xyz(lane, x, y, z);
    }
  };
  for (int64_t grp = (int64_t)blockIdx.x * wpb + warp; grp < n_groups; grp += stride) {
    double x, y, z;
    fetch(grp, x, y, z);
    eval_walkers<NS, NMO, EL, X, false, DERIV, EEN, 0, BF, FUSE>(P, sExp, sC, sDet, ws, x, y, z, lane, 0, 1, DerivOut{io.O, grp * G, io.M});
    bool flagged = false;
    if (lane < G) {
      const int64_t wo = grp * G + lane;
      if (wo < io.M) {
        const double *res = ws + GE::oResC(CP) + lane * 4;
        if (io.logpsi) io.logpsi[wo] = res[0];
        if (io.sign) io.sign[wo] = res[1];
        if (EL && io.eloc) io.eloc[wo] = res[2];
        flagged = res[3] != 0.0;
      }
    }
    // walkers whose reference determinant is nearly singular go to the explicit kernel
    int idx = -1;
    if (EL && io.fb_list) {
      const unsigned any = __ballot_sync(0xffffffffu, flagged);
      if (any && lane == 0) {
        idx = atomicAdd(io.fb_count, 1);
        io.fb_list[idx] = (int)grp;
        io.fb_done[idx] = 0;
      }
      if (FUSE) idx = __shfl_sync(0xffffffffu, idx, 0);
    }
    if (FUSE) {
      // rows in kernel order: Jastrow entries are final, the CI entries hold D_n / D_0 and want 1 / (Sigma / D_0)
      const double *res = ws + GE::oResC(CP);
      const double *sIden = sO + (G + 2) * np;
      const int nj = kJastrowParams + 7 * P.n_een;
      if (idx >= 0) {  // E_L of this group is still to be corrected: park its rows for the final kernel
        if (idx < io.fb_cap) {
          for (int wg = 0; wg < G; ++wg)
            if (grp * G + wg < io.M) {
              const double iden = sIden[wg];
              for (int p = lane; p < np; p += 32) io.fb_O[((int64_t)idx * G + wg) * np + p] = sO[wg * np + p] * ((p >= nj) ? iden : 1.0);
            }
        } else if (lane == 0) {
          *io.fb_over = 1;
        }
      } else {
        const int nw = (int)min((int64_t)G, io.M - grp * G);  // walkers of this group (the last one may be ragged)
        for (int p = lane; p < np; p += 32) {
          double so = 0.0, soe = 0.0;
          for (int wg = 0; wg < nw; ++wg) {
            const double v = sO[wg * np + p] * ((p >= nj) ? sIden[wg] : 1.0);
            so += v;
            soe = fma(v, res[wg * 4 + 2], soe);
          }
          accO[p] += so;
          accOE[p] += soe;
        }
        for (int wg = 0; wg < nw; ++wg) accE += res[wg * 4 + 2];  // every lane keeps the same sum
      }
    }
    __syncwarp();
  }
  if (FUSE) {
    // transposed, [2 n_param + 1][grid warps], so that the final kernel reads each parameter's column contiguously
    const int64_t nwarps = (int64_t)gridDim.x * wpb, me = (int64_t)blockIdx.x * wpb + warp;
    for (int p = lane; p < 2 * np; p += 32) io.fuse_part[p * nwarps + me] = accO[p];
    if (lane == 0) io.fuse_part[(int64_t)2 * np * nwarps + me] = accE;
  }
}

// Explicit re-evaluation of the groups listed by the fast kernel (rare; see kFallbackK).
// Work item = (listed group, determinant slice): the determinants of a group are dealt over SL warps of
// the whole grid, every warp rebuilds the MO rows of its group, eliminates its determinants and stores
// its partial sums; the warp that finishes a group last adds the partials in slice order (deterministic)
// and writes the outputs.
template <int NS, int NMO, bool X, int WPB, bool EEN = false>
__global__ void __launch_bounds__(WPB * 32, QMC_MINBLOCKS_EL)
    explicit_energy_kernel(const __grid_constant__ SysParams P, const WalkerIO io) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int n_list = *io.fb_count;
  if (n_list == 0) return;
  const int total_warps = (int)gridDim.x * WPB;
  int SL = total_warps / n_list;                       // slices per group
  SL = min(SL, (P.n_det_all + 3) / 4);                 // at least ~4 determinants per slice
  SL = max(SL, 1);
  const int64_t n_items = (int64_t)n_list * SL;
  // items are dealt block-first (item = round * grid + block), so few items spread over many SMs
  if ((int64_t)blockIdx.x >= n_items) return;          // nothing for this block: skip the constants
  const double *sC;
  const double *sExp;
  const DetRec *sDet;
  double *wsBase;
  load_constants<NMO>(P, smem, sC, sExp, sDet, wsBase);
  using GE = Geo<NS, NMO>;
  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;  // shfl: tells the compiler it is warp-uniform
  double *ws = wsBase + warp * GE::total;
  const int ne = X ? 2 * NS : P.n_e, G = X ? GE::GMAX : P.G;
  const int g = lane / ne, e = lane - g * ne;
  for (int64_t item = (int64_t)warp * gridDim.x + blockIdx.x; item < n_items; item += total_warps) {
    const int entry = (int)(item / SL), slice = (int)(item - (int64_t)entry * SL);
    const int64_t grp = io.fb_list[entry];
    const int64_t w = grp * G + g;
    double x, y, z;
    if ((g < G) && (w < io.M)) {
      x = io.r_in[((int64_t)e * 3 + 0) * io.M + w];
      y = io.r_in[((int64_t)e * 3 + 1) * io.M + w];
      z = io.r_in[((int64_t)e * 3 + 2) * io.M + w];
    } else {
      dummy_xyz(lane, x, y, z);
    }
    eval_walkers<NS, NMO, true, X, true, false, EEN>(P, sExp, sC, sDet, ws, x, y, z, lane, slice, SL);
    const double *res = ws + GE::oRes + (lane < G ? lane : 0) * 4;  // {Sigma, Sum d D t, J, energy share}
    if (lane < G) {
      io.fb_part[(item * G + lane) * 2 + 0] = res[0];   // eq. 4
      io.fb_part[(item * G + lane) * 2 + 1] = res[1];   // F.2 / F.4 with G.7
    }
    __threadfence();
    __syncwarp();  // every lane's partial is stored and fenced before lane 0 publishes the slice as done
    int last = 0;
    if (lane == 0) last = (atomicAdd(io.fb_done + entry, 1) == SL - 1) ? 1 : 0;
    last = __shfl_sync(0xffffffffu, last, 0);
    if (last) {
      __threadfence();
      // slice-ordered sums, the slices dealt over the lanes (fixed tree: deterministic); lane gw keeps walker gw
      double sig = 0.0, numk = 0.0;
      for (int gw = 0; gw < G; ++gw) {
        double a = 0.0, b = 0.0;
        for (int sl = lane; sl < SL; sl += 32) {
          const double *pp = io.fb_part + (((int64_t)entry * SL + sl) * G + gw) * 2;
          a += __ldcg(pp);       // eq. 4
          b += __ldcg(pp + 1);   // F.2 / F.4 with G.7
        }
        for (int m = 16; m > 0; m >>= 1) {
          a += shfl_xor_d(a, m);
          b += shfl_xor_d(b, m);
        }
        if (lane == gw) { sig = a; numk = b; }
      }
      const int64_t wo = grp * G + lane;
      if (lane < G && wo < io.M) {
        if (io.logpsi) io.logpsi[wo] = res[2] + log(fabs(sig));
        if (io.sign) io.sign[wo] = (sig > 0.0) ? 1.0 : ((sig < 0.0) ? -1.0 : 0.0);
        if (io.eloc) io.eloc[wo] = res[3] + numk / sig + P.vnn;
      }
    }
    __syncwarp();
  }
}

// ---------------------------------------------------------------------------------
// Orbital-parameter derivatives (eq. 6 factors of the AO and MO layers):
//   dC[w][beta][alpha] = d ln Psi / d C[beta][alpha] = sum_i phi_beta(r_i) Gamma[i][alpha]
//   dzeta[w][beta]     = d ln Psi / d zeta_beta      = sum_alpha C[beta][alpha] sum_i (d phi_beta / d zeta)(r_i) Gamma[i][alpha]
// with Gamma = d ln Sigma / d Phi from the reference's excitation tables (eval_walkers<..., ORB = 2>: A0^-1, T and
// Y = d(Sigma/D0)/dT; explicit per-determinant inverses, ORB = 1, for flagged walkers and general determinants), then
// a second pass over the shells that rebuilds phi and d phi / d zeta = phi (d ln N / d zeta - r) in the AO tile and
// contracts them with Gamma.  Outputs travel in io.logpsi (dC) and io.eloc (dzeta); either may be null.
// ---------------------------------------------------------------------------------
// Backflow coordinates of the lane's electron: rt_i = r_i + w sum_{j != i} (r_i - r_j) / r_ij over the other
// electrons of its walker (walker g of the warp, electron e); the first 96 doubles of the warp's scratch must be free.
__device__ __forceinline__ void backflow_lane_coords(double w, double *__restrict__ ws, int lane, int g, int e, int ne, double x,
                                                     double y, double z, double &xo, double &yo, double &zo) {
  ws[lane] = x; ws[32 + lane] = y; ws[64 + lane] = z;
  __syncwarp();
  const int base = g * ne;
  double px = 0.0, py = 0.0, pz = 0.0;
  for (int o = 1; o < ne; ++o) {
    int j = e + o;
    j -= (j >= ne) ? ne : 0;
    const double ddx = x - ws[base + j], ddy = y - ws[32 + base + j], ddz = z - ws[64 + base + j];
    const double ri = rsqrt_fast(fma(ddx, ddx, fma(ddy, ddy, ddz * ddz)));
    px = fma(ddx, ri, px); py = fma(ddy, ri, py); pz = fma(ddz, ri, pz);
  }
  xo = fma(w, px, x); yo = fma(w, py, y); zo = fma(w, pz, z);
  __syncwarp();
}

#ifndef QMC_NUC_DIRECT
#define QMC_NUC_DIRECT 1
#endif
#ifndef QMC_FRC_DIRECT
#define QMC_FRC_DIRECT 1
#endif
constexpr bool kFrcDirect = QMC_FRC_DIRECT != 0;  // nuclear energy gradient: the direct form of the second pass (0: the tile form)
constexpr bool kNucDirect = QMC_NUC_DIRECT != 0;  // nuclear log-gradient: the direct form of orbital_second_pass (0: the tile form)

// The second pass of the orbital-derivative kernels for group grp, with the normalised Gamma [G][ne][NMO] of its walkers in
// the warp's scratch (ws + oGam) and the lane's orbital position (xo, yo, zo): rebuilds phi and d phi / d zeta (nuclear mode:
// d phi / d R) in the AO tile and contracts them with Gamma on the FP64 tensor cores.
template <int NS, int NMO, bool X, bool NUC>
__device__ __forceinline__ void orbital_second_pass(const SysParams &P, const WalkerIO &io, double *__restrict__ ws,
                                                    const double *__restrict__ sC, const double *__restrict__ sExp, int lane,
                                                    int64_t grp, double xo, double yo, double zo) {
  using GE = Geo<NS, NMO>;
  constexpr int S = GE::S2, NT = GE::NT;
  constexpr bool nuc = NUC;
  const int ne = X ? 2 * NS : P.n_e, G = X ? GE::GMAX : P.G;
  double *dC = io.logpsi, *dZ = io.eloc, *dRo = io.O;
  const int *row_atom = P.ao_orig + P.n_chunks * kChunk;
  double *sGam = ws + GE::oGam;
  if constexpr (NUC && kNucDirect) {
    // Nuclear mode, direct form: dR[a][c] -= sum_i sum_{beta on a} w_i,beta d_c phi_beta(r_i) with w_i,beta = sum_alpha Gamma[i][alpha]
    // (N C)[beta][alpha].  Lane = electron: its Gamma row in registers, ONE pass over the shell records with all three
    // gradient components of every AO, the (N C) row read as broadcasts, per-centre sums in registers, summed over the
    // walker's electrons by shuffles where the centre changes.  (The tile form ran the pass twice and contracted both
    // column sets on the tensor cores: 0.57 ms per 32768 CO walkers against 0.46 for this one.)
    const int g = lane / ne;
    const bool act = lane < G * ne;
    double gam[NMO];
#pragma unroll
    for (int c = 0; c < NMO; ++c) gam[c] = (act && c < P.n_mo) ? sGam[lane * NMO + c] : 0.0;
    int chunk = 0, cur = -1;
    double dx = 0.0, dy = 0.0, dz = 0.0, r2 = 1.0, r = 1.0;
    double ax = 0.0, ay = 0.0, az = 0.0;
    auto flush_centre = [&]() {  // sum over the walker's electrons (lanes g ne .. g ne + ne - 1), electron 0 subtracts
      const int base = (act ? g : 0) * ne;
      double tx = 0.0, ty = 0.0, tz = 0.0;
      for (int j = 0; j < ne; ++j) {
        tx += shfl_d(ax, base + j, 32);
        ty += shfl_d(ay, base + j, 32);
        tz += shfl_d(az, base + j, 32);
      }
      const int64_t wo = grp * G + g;
      if (act && lane == base && wo < io.M && cur >= 0) {
        double *o = dRo + (wo * P.n_atoms + cur) * 3;
        o[0] -= tx; o[1] -= ty; o[2] -= tz;
      }
      ax = ay = az = 0.0;
    };
    for (int s = 0; s < P.n_shell; ++s) {
      const ShellRec &sh = P.shells[s];
      const int meta = sh.meta, kind = meta & 15;
      if (kind == SH_POW) continue;
      if (kind == SH_ATOM) {
        dx = xo - sh.zeta;
        dy = yo - sh.c1;
        dz = zo - sh.c2;
        r2 = fma(dx, dx, fma(dy, dy, dz * dz));
        r = r2 * rsqrt_fast(r2);
        continue;
      }
      double gr = exp_neg(-sh.zeta * r, sExp, P.mc);
      if (meta & kMetaK1) gr *= r;
      if (meta & kMetaK2) gr *= r2;
      const double rad0 = sh.kd / r2 - sh.zeta / r;  // phi = ang r^k e^{-zeta r}: d phi / d r_c = gr d ang / d d_c + phi rad0 d_c
      const int row = (meta >> 12) & 15, m = (meta >> 8) & 15;
      double ang[5], gx[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, gy[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, gz[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      int nf = 1;
      if (kind == SH_S) {
        ang[0] = 1.0;
      } else if (kind == SH_P) {
        ang[0] = dx; ang[1] = dy; ang[2] = dz; nf = 3;
        gx[0] = 1.0; gy[1] = 1.0; gz[2] = 1.0;
      } else if (kind == SH_P1) {
        ang[0] = (m == 0) ? dx : ((m == 1) ? dy : dz);
        gx[0] = (m == 0) ? 1.0 : 0.0; gy[0] = (m == 1) ? 1.0 : 0.0; gz[0] = (m == 2) ? 1.0 : 0.0;
      } else {
        // {xy, yz, zx, x^2 - y^2, 2 z^2 - x^2 - y^2} and their gradients
        const double dd[5] = {dx * dy, dy * dz, dz * dx, fma(dx, dx, -dy * dy), fma(2.0 * dz, dz, -fma(dx, dx, dy * dy))};
        const double hx[5] = {dy, 0.0, dz, 2.0 * dx, -2.0 * dx};
        const double hy[5] = {dx, dz, 0.0, -2.0 * dy, -2.0 * dy};
        const double hz[5] = {0.0, dy, dx, 0.0, 4.0 * dz};
        if (kind == SH_D) {
#pragma unroll
          for (int t = 0; t < 5; ++t) { ang[t] = dd[t]; gx[t] = hx[t]; gy[t] = hy[t]; gz[t] = hz[t]; }
          nf = 5;
        } else {
          const int mm = m < 5 ? m : 0;
          ang[0] = dd[mm]; gx[0] = hx[mm]; gy[0] = hy[mm]; gz[0] = hz[mm];
        }
      }
      const double *cfr = sC + chunk * ((kChunk / 4) * NT * 32);
#pragma unroll
      for (int t = 0; t < 5; ++t) {
        if (t < nf) {
          const int rw = row + t, R = chunk * kChunk + rw;
          const int at = row_atom[R];
          if (at != cur) {  // uniform: every lane walks the same records
            if (cur >= 0) flush_centre();
            cur = at;
          }
          double wgt = 0.0;
#pragma unroll
          for (int c = 0; c < NMO; ++c)
            wgt = fma(gam[c], cfr[(((rw >> 2) * NT) + (c >> 3)) * 32 + 4 * (c & 7) + (rw & 3)], wgt);
          const double phi = gr * ang[t], pr = phi * rad0;
          ax = fma(wgt, fma(gr, gx[t], pr * dx), ax);
          ay = fma(wgt, fma(gr, gy[t], pr * dy), ay);
          az = fma(wgt, fma(gr, gz[t], pr * dz), az);
        }
      }
      if (meta >> 20) ++chunk;
    }
    if (cur >= 0) flush_centre();
    __syncwarp();
    return;
  }
  {
    // second pass over the shells: phi into column lane, d phi / d zeta into column opCol(lane) of the tile
    double *const tile = ws;
    double *const tl = tile + lane, *const tz = tile + GE::opCol(lane);
    for (int pass = 0; pass < (nuc ? 2 : 1); ++pass) {
    const int comp = pass + 1;  // nuclear mode: component of the operator columns (y, then z); x rides in the phi columns of pass 0
    int chunk = 0;
    double dx = 0.0, dy = 0.0, dz = 0.0, r2 = 1.0, r = 1.0;
    for (int s = 0; s < P.n_shell; ++s) {
      const ShellRec &sh = P.shells[s];
      const int meta = sh.meta, kind = meta & 15;
      if (kind == SH_POW) continue;  // the radial power is in the shell records' own meta word
      if (kind == SH_ATOM) {
        dx = xo - sh.zeta;
        dy = yo - sh.c1;
        dz = zo - sh.c2;
        r2 = fma(dx, dx, fma(dy, dy, dz * dz));
        r = r2 * rsqrt_fast(r2);
        continue;
      }
      double gr = exp_neg(-sh.zeta * r, sExp, P.mc);
      if (meta & kMetaK1) gr *= r;
      if (meta & kMetaK2) gr *= r2;
      const double zf = sh.dlnN - r;  // d ln phi / d zeta
      // nuclear mode: phi = ang(d) r^k e^{-zeta r}, d phi / d r_c = gr d ang / d d_c + ang gr (k / r^2 - zeta / r) d_c
      const double dcmp = (comp == 0) ? dx : ((comp == 1) ? dy : dz);
      const double rad0 = sh.kd / r2 - sh.zeta / r;
      const double radc = rad0 * dcmp, radx = rad0 * dx;
      const int row = (meta >> 12) & 15, m = (meta >> 8) & 15;
      double ang[5], dang[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, dax[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      int nf = 1;
      if (kind == SH_S) {
        ang[0] = 1.0;
      } else if (kind == SH_P) {
        ang[0] = dx; ang[1] = dy; ang[2] = dz; nf = 3;
        dang[1] = (comp == 1) ? 1.0 : 0.0; dang[2] = (comp == 2) ? 1.0 : 0.0;
        dax[0] = 1.0;
      } else if (kind == SH_P1) {
        ang[0] = (m == 0) ? dx : ((m == 1) ? dy : dz);
        dang[0] = (m == comp) ? 1.0 : 0.0;
        dax[0] = (m == 0) ? 1.0 : 0.0;
      } else {
        const double dd[5] = {dx * dy, dy * dz, dz * dx, fma(dx, dx, -dy * dy), fma(2.0 * dz, dz, -fma(dx, dx, dy * dy))};
        // gradients of {xy, yz, zx, x^2 - y^2, 2 z^2 - x^2 - y^2}
        const double gd[5] = {(comp == 1) ? dx : 0.0, (comp == 1) ? dz : dy, (comp == 1) ? 0.0 : dx,
                              (comp == 1) ? -2.0 * dy : 0.0, (comp == 1) ? -2.0 * dy : 4.0 * dz};
        const double gx[5] = {dy, 0.0, dz, 2.0 * dx, -2.0 * dx};
        if (kind == SH_D) {
#pragma unroll
          for (int t = 0; t < 5; ++t) { ang[t] = dd[t]; dang[t] = gd[t]; dax[t] = gx[t]; }
          nf = 5;
        } else {
          ang[0] = dd[m < 5 ? m : 0];
          dang[0] = gd[m < 5 ? m : 0];
          dax[0] = gx[m < 5 ? m : 0];
        }
      }
#pragma unroll
      for (int t = 0; t < 5; ++t) {  // unrolled: ang / dang / dax stay in registers
        if (t < nf) {
          const double phi = gr * ang[t];
          tl[(row + t) * S] = nuc ? fma(gr, dax[t], phi * radx) : phi;
          tz[(row + t) * S] = nuc ? fma(gr, dang[t], phi * radc) : phi * zf;
        }
      }
      const int flush = meta >> 20;
      if (flush) {
        for (int pr = flush; pr < kChunk; ++pr) { tl[pr * S] = 0.0; tz[pr * S] = 0.0; }
        __syncwarp();
        // kernel-order (N C)[R][col] from the DMMA B-fragment table: [chunk][k-step][MO tile][4 n + k]
        const double *cfr = sC + chunk * ((kChunk / 4) * NT * 32);
        if (!nuc) {
          // Parameter mode on the FP64 tensor cores: per walker, D[AO row][MO] = sum_i tile[AO row][electron i] Gamma[i][MO]
          // with mma.m8n8k4 -- A fragments straight from the tile (rows = AO rows, k = the walker's electrons, four at a
          // time; columns past the walker's last electron meet zero rows of B), B fragments from Gamma, the D fragments
          // scaled and written out: dC from the value columns, dzeta = sum_MO (N C)[row][MO] D_zeta[row][MO] from the
          // operator columns (reduced over the four lanes that share a row).
          const int fr = lane >> 2, fk = lane & 3;
          constexpr int KS = (2 * NS + 3) / 4;
          for (int gg = 0; gg < G; ++gg) {
            const int64_t wo = grp * G + gg;
            double accv[2][NT][2], accz[2][NT][2];
#pragma unroll
            for (int m = 0; m < 2; ++m)
#pragma unroll
              for (int t = 0; t < NT; ++t) accv[m][t][0] = accv[m][t][1] = accz[m][t][0] = accz[m][t][1] = 0.0;
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
              const int ie = 4 * ks + fk;                        // electron of this lane's A column / B row
              const int iec = (ie < ne) ? ie : (ne - 1);         // any finite tile cell where B is zero
              double bfr[NT];
#pragma unroll
              for (int t = 0; t < NT; ++t) {
                const int col = 8 * t + fr;                      // B fragment: lane 4 n + k holds B[k][n]
                bfr[t] = (ie < ne && col < NMO) ? sGam[(gg * ne + ie) * NMO + col] : 0.0;
              }
#pragma unroll
              for (int m = 0; m < 2; ++m) {
                const double av = tile[(8 * m + fr) * S + gg * ne + iec];
                const double az = tile[(8 * m + fr) * S + GE::opCol(gg * ne + iec)];
#pragma unroll
                for (int t = 0; t < NT; ++t) {
                  dmma884(accv[m][t][0], accv[m][t][1], av, bfr[t]);
                  dmma884(accz[m][t][0], accz[m][t][1], az, bfr[t]);
                }
              }
            }
            // D fragment: lane 4 r + k holds D[r][2k], D[r][2k + 1]
#pragma unroll
            for (int m = 0; m < 2; ++m) {
              const int rw = 8 * m + fr, R = chunk * kChunk + rw, beta = P.ao_orig[R];
              double zsum = 0.0;
#pragma unroll
              for (int t = 0; t < NT; ++t)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                  const int col = 8 * t + 2 * fk + j;
                  if (col < NMO && col < P.n_mo) {
                    const double cf = cfr[(((rw >> 2) * NT) + (col >> 3)) * 32 + 4 * (col & 7) + (rw & 3)];
                    zsum = fma(cf, accz[m][t][j], zsum);
                    if (dC && beta >= 0 && wo < io.M)
                      dC[(wo * P.n_ao + beta) * P.n_mo_all + P.mo_orig[col]] = P.ao_nrm[R] * accv[m][t][j];
                  }
                }
              zsum += shfl_xor_d(zsum, 1);
              zsum += shfl_xor_d(zsum, 2);
              if (dZ && fk == 0 && beta >= 0 && wo < io.M) dZ[wo * P.n_ao + beta] = zsum;
            }
          }
          __syncwarp();
          ++chunk;
          continue;
        }
        {
          // Nuclear mode on the FP64 tensor cores: the same contraction on both column sets (pass 0: d/dx in the value
          // columns, d/dy in the operator columns; pass 1: d/dz in the operator columns), each D row multiplied by its
          // (N C) row and summed over the MOs, the row sums parked in the (now dead) tile, then one lane per (walker,
          // column set) adds the rows of each centre in row order and subtracts them from dR: the same lane owns the same
          // output in every chunk and pass, so its read-modify-writes are ordered.
          const int fr = lane >> 2, fk = lane & 3;
          constexpr int KS = (2 * NS + 3) / 4;
          double rs[2][GE::GMAX][2];  // [column set][walker][M-tile]
#pragma unroll
          for (int gg = 0; gg < GE::GMAX; ++gg) {
            rs[0][gg][0] = rs[0][gg][1] = rs[1][gg][0] = rs[1][gg][1] = 0.0;
            if (gg < G) {
              double accv[2][NT][2], accz[2][NT][2];
#pragma unroll
              for (int m = 0; m < 2; ++m)
#pragma unroll
                for (int t = 0; t < NT; ++t) accv[m][t][0] = accv[m][t][1] = accz[m][t][0] = accz[m][t][1] = 0.0;
#pragma unroll
              for (int ks = 0; ks < KS; ++ks) {
                const int ie = 4 * ks + fk;
                const int iec = (ie < ne) ? ie : (ne - 1);
                double bfr[NT];
#pragma unroll
                for (int t = 0; t < NT; ++t) {
                  const int col = 8 * t + fr;
                  bfr[t] = (ie < ne && col < NMO) ? sGam[(gg * ne + ie) * NMO + col] : 0.0;
                }
#pragma unroll
                for (int m = 0; m < 2; ++m) {
                  const double av = tile[(8 * m + fr) * S + gg * ne + iec];
                  const double az = tile[(8 * m + fr) * S + GE::opCol(gg * ne + iec)];
#pragma unroll
                  for (int t = 0; t < NT; ++t) {
                    if (pass == 0) dmma884(accv[m][t][0], accv[m][t][1], av, bfr[t]);
                    dmma884(accz[m][t][0], accz[m][t][1], az, bfr[t]);
                  }
                }
              }
#pragma unroll
              for (int m = 0; m < 2; ++m) {
                const int rw = 8 * m + fr;
                double sv = 0.0, sz = 0.0;
#pragma unroll
                for (int t = 0; t < NT; ++t)
#pragma unroll
                  for (int j2 = 0; j2 < 2; ++j2) {
                    const int col = 8 * t + 2 * fk + j2;
                    if (col < NMO && col < P.n_mo) {
                      const double cf = cfr[(((rw >> 2) * NT) + (col >> 3)) * 32 + 4 * (col & 7) + (rw & 3)];
                      sv = fma(cf, accv[m][t][j2], sv);
                      sz = fma(cf, accz[m][t][j2], sz);
                    }
                  }
                sv += shfl_xor_d(sv, 1); sv += shfl_xor_d(sv, 2);
                sz += shfl_xor_d(sz, 1); sz += shfl_xor_d(sz, 2);
                rs[0][gg][m] = sv;
                rs[1][gg][m] = sz;
              }
            }
          }
          __syncwarp();  // every lane is done reading the tile: park the row sums [column set][walker][16 rows] in it
          if (fk == 0) {
#pragma unroll
            for (int gg = 0; gg < GE::GMAX; ++gg)
              if (gg < G) {
#pragma unroll
                for (int m = 0; m < 2; ++m) {
                  tile[(0 * G + gg) * kChunk + 8 * m + fr] = rs[0][gg][m];
                  tile[(1 * G + gg) * kChunk + 8 * m + fr] = rs[1][gg][m];
                }
              }
          }
          __syncwarp();
          for (int item = lane; item < 2 * G; item += 32) {
            const int cset = item / G, gg = item - cset * G;
            const int64_t wo = grp * G + gg;
            if ((cset == 0 && pass != 0) || wo >= io.M) continue;
            const int cidx = (cset == 0) ? 0 : comp;
            double racc = 0.0;
            int cur = -1;
            for (int rw = 0; rw < kChunk; ++rw) {
              const int R = chunk * kChunk + rw;
              if (P.ao_orig[R] < 0) continue;
              const int at = row_atom[R];
              if (at != cur) {
                if (cur >= 0) dRo[(wo * P.n_atoms + cur) * 3 + cidx] -= racc;
                cur = at;
                racc = 0.0;
              }
              racc += tile[(cset * G + gg) * kChunk + rw];
            }
            if (cur >= 0) dRo[(wo * P.n_atoms + cur) * 3 + cidx] -= racc;
          }
        }
        __syncwarp();
        ++chunk;
      }
    }
    __syncwarp();
    }
  }
}

// BF: backflow wavefunction: phi, d phi / d zeta and d phi / d R are evaluated at the backflow coordinates, which
// depend on none of these parameters; Gamma from the values-only evaluator at the same coordinates.
template <int NS, int NMO, bool X, int WPB, bool NUC = false, bool BF = false>
__global__ void __launch_bounds__(WPB * 32, 1)
    orbital_derivatives_kernel(const __grid_constant__ SysParams P, const WalkerIO io) {
  extern __shared__ __align__(16) unsigned char smem[];
  const double *sC;
  const double *sExp;
  const DetRec *sDet;
  double *wsBase;
  load_constants<NMO>(P, smem, sC, sExp, sDet, wsBase);
  using GE = Geo<NS, NMO>;
  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
  double *ws = wsBase + warp * (GE::total + GE::orbExtra);
  const int ne = X ? 2 * NS : P.n_e, G = X ? GE::GMAX : P.G;
  const int g = lane / ne, e = lane - g * ne;
  const int64_t n_groups = (io.M + G - 1) / G;
  // nuclear mode (qmc_nuclear_log_gradient): io.O = dR [M][n_atoms][3]; d phi / d R_c = -d phi / d r_c takes the place of
  // phi and d phi / d zeta in the two column sets of the tile: the second pass runs twice, (x, y) then z, and the
  // contraction is summed over the rows of each centre
  // The groups are dealt by an atomic counter (io.fb_count, zeroed by the host): a group on the explicit route costs tens of
  // ordinary ones, and where such groups sit at regular distances a fixed assignment piles them onto the same warps
  // (measured: 0.53 ms with 10 warps per block, 0.74 ms with 9 or 12 on the same walkers).
  auto next_group = [&]() {
    int v = 0;
    if (lane == 0) v = atomicAdd(io.fb_count, 1);
    return (int64_t)__shfl_sync(0xffffffffu, v, 0);
  };
  for (int64_t grp = next_group(); grp < n_groups; grp = next_group()) {
    const int64_t w = grp * G + g;
    double x, y, z;
    if ((g < G) && (w < io.M)) {
      x = io.r_in[((int64_t)e * 3 + 0) * io.M + w];
      y = io.r_in[((int64_t)e * 3 + 1) * io.M + w];
      z = io.r_in[((int64_t)e * 3 + 2) * io.M + w];
    } else {
      dummy_xyz(lane, x, y, z);
    }
    // Gamma = d ln Sigma / d Phi from the reference's tables (one elimination per spin); when a walker of the group
    // has (Sigma/D_0)^2 > kFallbackOrb (reference near-singular) or the expansion has general determinants, from every
    // determinant's inverse instead: unnormalised Gamma and Sigma (sRes[4 g])
    double xo = x, yo = y, zo = z;  // where this lane's orbitals sit
    if (BF) backflow_lane_coords(P.bf_w, ws, lane, (lane < G * ne) ? g : 0, e, ne, x, y, z, xo, yo, zo);
    bool expl = P.n_gen > 0;
    if (!expl) {
      eval_walkers<NS, NMO, false, X, false, false, false, 2, BF>(P, sExp, sC, sDet, ws, x, y, z, lane, 0, 1);
      for (int gg = 0; gg < G; ++gg) {
        const double den = (ws + GE::oProb)[gg * 8 + 3];  // Sigma / D_0 of walker gg (NaN for a singular reference)
        const double kap = (ws + GE::oProb)[gg * 8 + 7];  // max |T| over both spins
        expl |= !(den * den <= kFallbackOrb) || !(kap * kap <= kFallbackOrbKappa);
      }
      __syncwarp();
    }
    if (expl) {  // listed for orbital_explicit_kernel, which deals the determinants of such a group over several warps
      if (lane == 0) {
        const int idx = atomicAdd(io.fb_count + 1, 1);
        io.fb_list[idx] = (int)grp;
        io.fb_done[idx] = 0;
      }
      __syncwarp();
      continue;
    }
    orbital_second_pass<NS, NMO, X, NUC>(P, io, ws, sC, sExp, lane, grp, xo, yo, zo);
  }
}

// The groups orbital_derivatives_kernel listed (a walker with a nearly singular reference, or an expansion with general
// determinants): Gamma from every determinant's own inverse.  Work item = (listed group, determinant slice), dealt over the
// whole grid as in explicit_energy_kernel: every warp rebuilds the MO rows of its group and accumulates the unnormalised
// Gamma and Sigma of its determinants; the warp that finishes a group last adds the partials in slice order
// (deterministic), normalises and runs the second pass.  (One warp per group took 100 determinants in a row while the rest
// of the grid waited: 0.19 of 0.53 ms for 32768 CO walkers.)
template <int NS, int NMO, bool X, int WPB, bool NUC = false, bool BF = false>
__global__ void __launch_bounds__(WPB * 32, 1)
    orbital_explicit_kernel(const __grid_constant__ SysParams P, const WalkerIO io) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int n_list = io.fb_count[1];
  if (n_list == 0) return;
  const int total_warps = (int)gridDim.x * WPB;
  int SL = total_warps / n_list;                       // slices per group
  SL = min(SL, (P.n_det_all + 3) / 4);                 // at least ~4 determinants per slice
  SL = max(SL, 1);
  const int64_t n_items = (int64_t)n_list * SL;
  if ((int64_t)blockIdx.x >= n_items) return;          // items are dealt block-first: nothing for this block
  const double *sC;
  const double *sExp;
  const DetRec *sDet;
  double *wsBase;
  load_constants<NMO>(P, smem, sC, sExp, sDet, wsBase);
  using GE = Geo<NS, NMO>;
  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
  double *ws = wsBase + warp * (GE::total + GE::orbExtra);
  const int ne = X ? 2 * NS : P.n_e, G = X ? GE::GMAX : P.G;
  const int g = lane / ne, e = lane - g * ne;
  double *sGam = ws + GE::oGam, *sRes = ws + GE::oRes;
  const int nG = G * ne * NMO, PS = nG + G;            // a partial record: Gamma [G][ne][NMO], then Sigma per walker
  for (int64_t item = (int64_t)warp * gridDim.x + blockIdx.x; item < n_items; item += total_warps) {
    const int entry = (int)(item / SL), slice = (int)(item - (int64_t)entry * SL);
    const int64_t grp = io.fb_list[entry];
    const int64_t w = grp * G + g;
    double x, y, z;
    if ((g < G) && (w < io.M)) {
      x = io.r_in[((int64_t)e * 3 + 0) * io.M + w];
      y = io.r_in[((int64_t)e * 3 + 1) * io.M + w];
      z = io.r_in[((int64_t)e * 3 + 2) * io.M + w];
    } else {
      dummy_xyz(lane, x, y, z);
    }
    double xo = x, yo = y, zo = z;
    if (BF) backflow_lane_coords(P.bf_w, ws, lane, (lane < G * ne) ? g : 0, e, ne, x, y, z, xo, yo, zo);
    eval_walkers<NS, NMO, false, X, true, false, false, 1, BF>(P, sExp, sC, sDet, ws, x, y, z, lane, slice, SL);
    int last = 1;
    if (SL > 1) {
      double *part = io.fb_part + item * PS;
      for (int i = lane; i < nG; i += 32) part[i] = sGam[i];
      if (lane < G) part[nG + lane] = sRes[lane * 4 + 0];
      __threadfence();
      __syncwarp();  // every lane's partial is stored and fenced before lane 0 publishes the slice as done
      int l = 0;
      if (lane == 0) l = (atomicAdd(io.fb_done + entry, 1) == SL - 1) ? 1 : 0;
      last = __shfl_sync(0xffffffffu, l, 0);
      if (last) {
        __threadfence();
        const double *p0 = io.fb_part + (int64_t)entry * SL * PS;
        for (int i = lane; i < nG; i += 32) {
          double a = 0.0;
          for (int sl = 0; sl < SL; ++sl) a += __ldcg(p0 + (int64_t)sl * PS + i);
          sGam[i] = a;
        }
        if (lane < G) {
          double a = 0.0;
          for (int sl = 0; sl < SL; ++sl) a += __ldcg(p0 + (int64_t)sl * PS + nG + lane);
          sRes[lane * 4 + 0] = a;
        }
        __syncwarp();
      }
    }
    if (last) {
      for (int i = lane; i < nG; i += 32) sGam[i] /= sRes[(i / (ne * NMO)) * 4 + 0];
      __syncwarp();
      orbital_second_pass<NS, NMO, X, NUC>(P, io, ws, sC, sExp, lane, grp, xo, yo, zo);
    }
    __syncwarp();
  }
}

#ifndef QMC_VARIANT_TU  // (the per-variant translation units hold only the template kernels)
// ---------------------------------------------------------------------------------
// Nuclear dependence of the Jastrow factor (eq. 7's grad_alpha ln rho): dR[w][a][c] = d J / d R_a,c
//   D.2: K(r_ia) = (w0 r + w1 r^2) / (1 + w2 r)              ->  -K' e_ai
//   D.3: c f(r_ai) g(r_aj) h(r_ij), ordered pairs i != j, c = c_mu / 2 (reading Q22)  ->  -c h (f' g e_ai + f g' e_aj)
// One thread per walker (SoA loads coalesce); writes every entry, zeros without those kernels.  The AO part is
// subtracted afterwards by orbital_derivatives_kernel in nuclear mode.
// ---------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
    nuclear_jastrow_gradient_kernel(const __grid_constant__ SysParams P, const double *__restrict__ rin, const int64_t M,
                                    double *__restrict__ dR) {
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= M) return;
  const int ne = P.n_e;
  for (int a = 0; a < P.n_atoms; ++a) {
    const double X = P.atom[a][0], Y = P.atom[a][1], Z = P.atom[a][2];
    double gx = 0.0, gy = 0.0, gz = 0.0;
    for (int i = 0; i < ne; ++i) {
      const double xi = rin[((int64_t)i * 3 + 0) * M + w], yi = rin[((int64_t)i * 3 + 1) * M + w],
                   zi = rin[((int64_t)i * 3 + 2) * M + w];
      const double ax = xi - X, ay = yi - Y, az = zi - Z;
      const double rai = sqrt(fma(ax, ax, fma(ay, ay, az * az)));
      if (P.has_en) {
        const double N = fma(P.en_w1 * rai, rai, P.en_w0 * rai), D = fma(P.en_w2, rai, 1.0);
        const double K1 = (fma(2.0 * P.en_w1, rai, P.en_w0) * D - N * P.en_w2) / (D * D * rai);
        gx = fma(-K1, ax, gx);
        gy = fma(-K1, ay, gy);
        gz = fma(-K1, az, gz);
      }
      if (P.n_een > 0)
        for (int j = 0; j < ne; ++j) {
          if (j == i) continue;
          const double xj = rin[((int64_t)j * 3 + 0) * M + w], yj = rin[((int64_t)j * 3 + 1) * M + w],
                       zj = rin[((int64_t)j * 3 + 2) * M + w];
          const double bx = xj - X, by = yj - Y, bz = zj - Z;
          const double ex = xi - xj, ey = yi - yj, ez = zi - zj;
          const double raj = sqrt(fma(bx, bx, fma(by, by, bz * bz))), rij = sqrt(fma(ex, ex, fma(ey, ey, ez * ez)));
          for (int mu = 0; mu < P.n_een; ++mu) {
            const double *q = P.een[mu];
            const double Df = fma(q[2], rai, 1.0), Dg = fma(q[4], raj, 1.0), Dh = fma(q[6], rij, 1.0);
            const double f = q[1] * rai / Df, f1 = q[1] / (Df * Df);
            const double g = q[3] * raj / Dg, g1 = q[3] / (Dg * Dg);
            const double ch = q[0] * q[5] * rij / Dh;
            const double ti = ch * f1 * g / rai, tj = ch * f * g1 / raj;
            gx -= fma(ti, ax, tj * bx);
            gy -= fma(ti, ay, tj * by);
            gz -= fma(ti, az, tj * bz);
          }
        }
    }
    double *o = dR + (w * P.n_atoms + a) * 3;
    o[0] = gx;
    o[1] = gy;
    o[2] = gz;
  }
}

#endif  // QMC_VARIANT_TU
// ---------------------------------------------------------------------------------
// Nuclear gradient of the local energy, grad_alpha E_L: the first term of the force estimator, eq. 7.
// The atomic positions are inputs of the AO layer: d phi_beta(r_i) / d R_alpha = -grad phi_beta(r_i)
// for the AOs of centre alpha.  With the Pade e-e Jastrow D.1 (which does not see the nuclei)
//   E_L = -1/2 (lap J + |grad J|^2) + K + V,   K = sum_n w_n t_n / sum_n w_n,  w_n = d_n D_n^up D_n^dn,
//   t_n = Tr(A_n^-1 B_n),  B = -1/2 lap phi - grad_i J . grad phi   (F.1-F.4, G.7 with the combined operator),
// and the chain rule through every determinant collapses into two weight matrices (electrons x MOs),
//   Gamma  = d Sigma / d Phi  = d (sum w t) / d B,      Gamma2 = d (sum w t) / d Phi   (eval_walkers<..., ORB = 3>):
//   d_j K = [ (Gamma2 - K Gamma) : d_j Phi + Gamma : d_j B ] / Sigma.
// At AO level, for a harmonic S (lap S = 0, grad S . d = l S), f = r^k e^{-zeta r}, u = d / r, rho = f'/f = k/r - zeta,
// F2 = f''/f = rho^2 - k/r^2, lambda = lap(S f)/(S f) = zeta^2 - c1/r + c2/r^2 (c1, c2 of the shell record),
// lambda' = c1/r^2 - 2 c2/r^3, q = grad_i J . u, gs = grad_i J . grad S, w_c = sum_e (grad_i J)_e S_ce:
//   -d_c phi = -f (S_c + S rho u_c)                                                              (value columns)
//   1/2 d_c lap phi + grad_i J . d_c grad phi = f [ S_c (lambda/2 + rho q) + w_c + S rho (grad_i J)_c / r
//        + u_c ( S (rho lambda + lambda')/2 + rho gs + S q (F2 - rho / r) ) ]                   (operator columns)
// One pass over the shell records per Cartesian component; the tile is contracted with the two weight matrices and
// the (N C) fragments and summed per centre.  d V / d R_alpha was written by nuclear_potential_gradient_kernel.
// This is the explicit route (every determinant eliminated on its own) for every walker.
// ---------------------------------------------------------------------------------
template <int CMP>
__device__ __forceinline__ void force_ao_pair(double f, double S, double Sx, double Sy, double Sz, double wc, double gs,
                                              double ux, double uy, double uz, double gJx, double gJy, double gJz, double ri,
                                              double rho, double q, double lam, double dlam, double F2, double &val, double &op) {
  const double Sc = (CMP == 0) ? Sx : ((CMP == 1) ? Sy : Sz);
  const double uc = (CMP == 0) ? ux : ((CMP == 1) ? uy : uz);
  const double gc = (CMP == 0) ? gJx : ((CMP == 1) ? gJy : gJz);
  val = -f * fma(S * rho, uc, Sc);
  const double inner = fma(0.5 * S, fma(rho, lam, dlam), fma(rho, gs, S * q * (F2 - rho * ri)));
  op = f * (fma(Sc, fma(rho, q, 0.5 * lam), wc) + fma(uc, inner, S * rho * gc * ri));
}

template <int NS, int NMO, bool X, int WPB>
__global__ void __launch_bounds__(WPB * 32, 1)
    nuclear_energy_gradient_kernel(const __grid_constant__ SysParams P, const WalkerIO io) {
  extern __shared__ __align__(16) unsigned char smem[];
  const double *sC;
  const double *sExp;
  const DetRec *sDet;
  double *wsBase;
  load_constants<NMO>(P, smem, sC, sExp, sDet, wsBase);
  using GE = Geo<NS, NMO>;
  constexpr int S = GE::S2, NT = GE::NT;
  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;
  double *ws = wsBase + warp * (GE::total + GE::frcExtra);
  const int ne = X ? 2 * NS : P.n_e, G = X ? GE::GMAX : P.G;
  const int g = lane / ne, e = lane - g * ne;
  const int64_t n_groups = (io.M + G - 1) / G;
  const int64_t stride = (int64_t)gridDim.x * WPB;
  double *dEo = io.O;  // [M][n_atoms][3], initialised with d V / d R
  const int *row_atom = P.ao_orig + P.n_chunks * kChunk;
  double *sGam = ws + GE::oGam, *sGam2 = ws + GE::oGam2;
  const double *sGJ = ws + GE::oGJ;
  const double *sRes = ws + GE::oRes;
  // groups dealt by an atomic counter (io.fb_count, zeroed by the host), as in orbital_derivatives_kernel
  auto next_group = [&]() {
    int v = 0;
    if (lane == 0) v = atomicAdd(io.fb_count, 1);
    return (int64_t)__shfl_sync(0xffffffffu, v, 0);
  };
  (void)stride;
  for (int64_t grp = next_group(); grp < n_groups; grp = next_group()) {
    const int64_t w = grp * G + g;
    double x, y, z;
    if ((g < G) && (w < io.M)) {
      x = io.r_in[((int64_t)e * 3 + 0) * io.M + w];
      y = io.r_in[((int64_t)e * 3 + 1) * io.M + w];
      z = io.r_in[((int64_t)e * 3 + 2) * io.M + w];
    } else {
      dummy_xyz(lane, x, y, z);
    }
    // The two weight matrices G1 (of d_j B) and G2 (of d_j Phi): from the reference's tables (one elimination per
    // spin, eval_walkers<..., ORB = 4>); for a group with a walker whose reference is nearly singular (the E_L flag, or
    // (Sigma/D_0)^2 > kFallbackOrb, kappa^2 > kFallbackOrbKappa) and for expansions with general determinants, from
    // every determinant's own elimination (ORB = 3): G1 = Gamma / Sigma, G2 = (Gamma2 - K Gamma) / Sigma.
    bool expl = P.n_gen > 0;
    if (!expl) {
      eval_walkers<NS, NMO, true, X, false, false, false, 4>(P, sExp, sC, sDet, ws, x, y, z, lane, 0, 1);
      const double *sProb = ws + GE::oProb;
      for (int gg = 0; gg < G; ++gg) {
        const double den = sProb[(2 * gg + 1) * 4 + 1], ku = sProb[(2 * gg) * 4 + 3], kd = sProb[(2 * gg + 1) * 4 + 3];
        expl |= (sRes[gg * 4 + 3] != 0.0) || !(den * den <= kFallbackOrb) || !(ku * ku <= kFallbackOrbKappa) ||
                !(kd * kd <= kFallbackOrbKappa);
      }
      __syncwarp();
    }
    if (expl) {
      eval_walkers<NS, NMO, true, X, true, false, false, 3>(P, sExp, sC, sDet, ws, x, y, z, lane, 0, 1);
      for (int i = lane; i < G * ne * NMO; i += 32) {
        const int gg = i / (ne * NMO);
        const double sig = sRes[gg * 4 + 0], K = sRes[gg * 4 + 1] / sig;
        const double g1 = sGam[i] / sig;
        sGam2[i] = sGam2[i] / sig - K * g1;
        sGam[i] = g1;
      }
    }
    const double gJx = sGJ[lane], gJy = sGJ[32 + lane], gJz = sGJ[64 + lane];
    __syncwarp();
    if (kFrcDirect) {
      // Direct form (as the nuclear log-gradient's): lane = electron with its rows of G1 and G2 in registers, ONE pass over
      // the shell records (exp once) with the value and operator tangents of all three components, the (N C) row read as
      // broadcasts: dE[a][c] += sum_{beta on a} (w2 val_c + w1 op_c), w1,2 = sum_alpha G1,2[i][alpha] (N C)[beta][alpha],
      // summed over the walker's electrons by shuffles where the centre changes.
      const bool act = lane < G * ne;
      double g1[NMO], g2[NMO];
#pragma unroll
      for (int c = 0; c < NMO; ++c) {
        g1[c] = (act && c < P.n_mo) ? sGam[lane * NMO + c] : 0.0;
        g2[c] = (act && c < P.n_mo) ? sGam2[lane * NMO + c] : 0.0;
      }
      int chunk = 0, cur = -1;
      double dx = 0.0, dy = 0.0, dz = 0.0, r2 = 1.0, r = 1.0, ri = 1.0, q = 0.0;
      double ax = 0.0, ay = 0.0, az = 0.0;
      auto flush_centre = [&]() {
        const int base = (act ? g : 0) * ne;
        double tx = 0.0, ty = 0.0, tz2 = 0.0;
        for (int j = 0; j < ne; ++j) {
          tx += shfl_d(ax, base + j, 32);
          ty += shfl_d(ay, base + j, 32);
          tz2 += shfl_d(az, base + j, 32);
        }
        const int64_t wo = grp * G + g;
        if (act && lane == base && wo < io.M && cur >= 0) {
          double *o = dEo + (wo * P.n_atoms + cur) * 3;
          o[0] += tx; o[1] += ty; o[2] += tz2;
        }
        ax = ay = az = 0.0;
      };
      for (int s = 0; s < P.n_shell; ++s) {
        const ShellRec &sh = P.shells[s];
        const int meta = sh.meta, kind = meta & 15;
        if (kind == SH_POW) continue;
        if (kind == SH_ATOM) {
          dx = x - sh.zeta;
          dy = y - sh.c1;
          dz = z - sh.c2;
          r2 = fma(dx, dx, fma(dy, dy, dz * dz));
          ri = rsqrt_fast(r2);
          r = r2 * ri;
          q = fma(gJx, dx, fma(gJy, dy, gJz * dz)) * ri;
          continue;
        }
        double f = exp_neg(-sh.zeta * r, sExp, P.mc);
        if (meta & kMetaK1) f *= r;
        if (meta & kMetaK2) f *= r2;
        const double ux = dx * ri, uy = dy * ri, uz = dz * ri;
        const double rho = fma(sh.kd, ri, -sh.zeta);
        const double F2 = fma(rho, rho, -sh.kd * ri * ri);
        const double lam = fma(fma(sh.c2, ri, -sh.c1), ri, sh.zeta * sh.zeta);
        const double dlam = fma(-2.0 * sh.c2, ri, sh.c1) * ri * ri;
        const int row = (meta >> 12) & 15, m = (meta >> 8) & 15;
        double Sv[5], Sx[5], Sy[5], Sz[5], wx[5], wy[5], wz[5];
        int nf = 1;
        Sv[0] = 1.0; Sx[0] = Sy[0] = Sz[0] = 0.0; wx[0] = wy[0] = wz[0] = 0.0;
        if (kind == SH_P || kind == SH_P1) {
          const double pv[3] = {dx, dy, dz};
          if (kind == SH_P) {
            nf = 3;
#pragma unroll
            for (int t = 0; t < 3; ++t) { Sv[t] = pv[t]; Sx[t] = (t == 0); Sy[t] = (t == 1); Sz[t] = (t == 2); wx[t] = wy[t] = wz[t] = 0.0; }
          } else {
            Sv[0] = (m == 0) ? dx : ((m == 1) ? dy : dz);
            Sx[0] = (m == 0); Sy[0] = (m == 1); Sz[0] = (m == 2);
          }
        } else if (kind == SH_D || kind == SH_D1) {
          const double dS[5] = {dx * dy, dy * dz, dz * dx, fma(dx, dx, -dy * dy), fma(2.0 * dz, dz, -fma(dx, dx, dy * dy))};
          const double dSx[5] = {dy, 0.0, dz, 2.0 * dx, -2.0 * dx};
          const double dSy[5] = {dx, dz, 0.0, -2.0 * dy, -2.0 * dy};
          const double dSz[5] = {0.0, dy, dx, 0.0, 4.0 * dz};
          const double dwx[5] = {gJy, 0.0, gJz, 2.0 * gJx, -2.0 * gJx};
          const double dwy[5] = {gJx, gJz, 0.0, -2.0 * gJy, -2.0 * gJy};
          const double dwz[5] = {0.0, gJy, gJx, 0.0, 4.0 * gJz};
          if (kind == SH_D) {
            nf = 5;
#pragma unroll
            for (int t = 0; t < 5; ++t) { Sv[t] = dS[t]; Sx[t] = dSx[t]; Sy[t] = dSy[t]; Sz[t] = dSz[t]; wx[t] = dwx[t]; wy[t] = dwy[t]; wz[t] = dwz[t]; }
          } else {
#pragma unroll
            for (int t = 0; t < 5; ++t)
              if (t == m) { Sv[0] = dS[t]; Sx[0] = dSx[t]; Sy[0] = dSy[t]; Sz[0] = dSz[t]; wx[0] = dwx[t]; wy[0] = dwy[t]; wz[0] = dwz[t]; }
          }
        }
        const double *cfr = sC + chunk * ((kChunk / 4) * NT * 32);
#pragma unroll
        for (int t = 0; t < 5; ++t) {
          if (t < nf) {
            const int rw = row + t, R = chunk * kChunk + rw;
            const int at = row_atom[R];
            if (at != cur) {  // uniform: every lane walks the same records
              if (cur >= 0) flush_centre();
              cur = at;
            }
            double w1 = 0.0, w2 = 0.0;
#pragma unroll
            for (int c = 0; c < NMO; ++c) {
              const double cf = cfr[(((rw >> 2) * NT) + (c >> 3)) * 32 + 4 * (c & 7) + (rw & 3)];
              w1 = fma(g1[c], cf, w1);
              w2 = fma(g2[c], cf, w2);
            }
            const double gs = fma(gJx, Sx[t], fma(gJy, Sy[t], gJz * Sz[t]));
            double val, op;
            force_ao_pair<0>(f, Sv[t], Sx[t], Sy[t], Sz[t], wx[t], gs, ux, uy, uz, gJx, gJy, gJz, ri, rho, q, lam, dlam, F2, val, op);
            ax = fma(w2, val, fma(w1, op, ax));
            force_ao_pair<1>(f, Sv[t], Sx[t], Sy[t], Sz[t], wy[t], gs, ux, uy, uz, gJx, gJy, gJz, ri, rho, q, lam, dlam, F2, val, op);
            ay = fma(w2, val, fma(w1, op, ay));
            force_ao_pair<2>(f, Sv[t], Sx[t], Sy[t], Sz[t], wz[t], gs, ux, uy, uz, gJx, gJy, gJz, ri, rho, q, lam, dlam, F2, val, op);
            az = fma(w2, val, fma(w1, op, az));
          }
        }
        if (meta >> 20) ++chunk;
      }
      if (cur >= 0) flush_centre();
      __syncwarp();
      continue;
    }
    double *const tile = ws;
    double *const tl = tile + lane, *const tz = tile + GE::opCol(lane);
#pragma unroll 1
    for (int cmp = 0; cmp < 3; ++cmp) {
      int chunk = 0;
      double dx = 0.0, dy = 0.0, dz = 0.0, r2 = 1.0, r = 1.0, ri = 1.0, q = 0.0;
      for (int s = 0; s < P.n_shell; ++s) {
        const ShellRec &sh = P.shells[s];
        const int meta = sh.meta, kind = meta & 15;
        if (kind == SH_POW) continue;  // the radial power is in the shell records' own meta word
        if (kind == SH_ATOM) {
          dx = x - sh.zeta;
          dy = y - sh.c1;
          dz = z - sh.c2;
          r2 = fma(dx, dx, fma(dy, dy, dz * dz));
          ri = rsqrt_fast(r2);
          r = r2 * ri;
          q = fma(gJx, dx, fma(gJy, dy, gJz * dz)) * ri;
          continue;
        }
        double f = exp_neg(-sh.zeta * r, sExp, P.mc);
        if (meta & kMetaK1) f *= r;
        if (meta & kMetaK2) f *= r2;
        const double ux = dx * ri, uy = dy * ri, uz = dz * ri;
        const double rho = fma(sh.kd, ri, -sh.zeta);
        const double F2 = fma(rho, rho, -sh.kd * ri * ri);
        const double lam = fma(fma(sh.c2, ri, -sh.c1), ri, sh.zeta * sh.zeta);
        const double dlam = fma(-2.0 * sh.c2, ri, sh.c1) * ri * ri;
        const int row = (meta >> 12) & 15, m = (meta >> 8) & 15;
        // harmonics of this record: S, grad S, w = Hess(S) grad_i J, gs = grad_i J . grad S
        double Sv[5], Sx[5], Sy[5], Sz[5], wx[5], wy[5], wz[5];
        int nf = 1;
        Sv[0] = 1.0; Sx[0] = Sy[0] = Sz[0] = 0.0; wx[0] = wy[0] = wz[0] = 0.0;
        if (kind == SH_P || kind == SH_P1) {
          const double pv[3] = {dx, dy, dz};
          if (kind == SH_P) {
            nf = 3;
#pragma unroll
            for (int t = 0; t < 3; ++t) { Sv[t] = pv[t]; Sx[t] = (t == 0); Sy[t] = (t == 1); Sz[t] = (t == 2); wx[t] = wy[t] = wz[t] = 0.0; }
          } else {
            Sv[0] = (m == 0) ? dx : ((m == 1) ? dy : dz);
            Sx[0] = (m == 0); Sy[0] = (m == 1); Sz[0] = (m == 2);
          }
        } else if (kind == SH_D || kind == SH_D1) {
          const double dS[5] = {dx * dy, dy * dz, dz * dx, fma(dx, dx, -dy * dy), fma(2.0 * dz, dz, -fma(dx, dx, dy * dy))};
          const double dSx[5] = {dy, 0.0, dz, 2.0 * dx, -2.0 * dx};
          const double dSy[5] = {dx, dz, 0.0, -2.0 * dy, -2.0 * dy};
          const double dSz[5] = {0.0, dy, dx, 0.0, 4.0 * dz};
          const double dwx[5] = {gJy, 0.0, gJz, 2.0 * gJx, -2.0 * gJx};
          const double dwy[5] = {gJx, gJz, 0.0, -2.0 * gJy, -2.0 * gJy};
          const double dwz[5] = {0.0, gJy, gJx, 0.0, 4.0 * gJz};
          if (kind == SH_D) {
            nf = 5;
#pragma unroll
            for (int t = 0; t < 5; ++t) { Sv[t] = dS[t]; Sx[t] = dSx[t]; Sy[t] = dSy[t]; Sz[t] = dSz[t]; wx[t] = dwx[t]; wy[t] = dwy[t]; wz[t] = dwz[t]; }
          } else {
#pragma unroll
            for (int t = 0; t < 5; ++t)
              if (t == m) { Sv[0] = dS[t]; Sx[0] = dSx[t]; Sy[0] = dSy[t]; Sz[0] = dSz[t]; wx[0] = dwx[t]; wy[0] = dwy[t]; wz[0] = dwz[t]; }
          }
        }
#pragma unroll
        for (int t = 0; t < 5; ++t) {
          if (t < nf) {
            const double gs = fma(gJx, Sx[t], fma(gJy, Sy[t], gJz * Sz[t]));
            double val, op;
            if (cmp == 0) force_ao_pair<0>(f, Sv[t], Sx[t], Sy[t], Sz[t], wx[t], gs, ux, uy, uz, gJx, gJy, gJz, ri, rho, q, lam, dlam, F2, val, op);
            else if (cmp == 1) force_ao_pair<1>(f, Sv[t], Sx[t], Sy[t], Sz[t], wy[t], gs, ux, uy, uz, gJx, gJy, gJz, ri, rho, q, lam, dlam, F2, val, op);
            else force_ao_pair<2>(f, Sv[t], Sx[t], Sy[t], Sz[t], wz[t], gs, ux, uy, uz, gJx, gJy, gJz, ri, rho, q, lam, dlam, F2, val, op);
            tl[(row + t) * S] = val;
            tz[(row + t) * S] = op;
          }
        }
        const int flush = meta >> 20;
        if (flush) {
          for (int pr = flush; pr < kChunk; ++pr) { tl[pr * S] = 0.0; tz[pr * S] = 0.0; }
          __syncwarp();
          const double *cfr = sC + chunk * ((kChunk / 4) * NT * 32);
          constexpr int CW = NMO <= 2 ? 2 : (NMO <= 4 ? 4 : (NMO <= 8 ? 8 : 16));
          for (int pi = lane; pi < ((G * CW + 31) & ~31); pi += 32) {
            const int gq = pi / CW, col = pi & (CW - 1);
            const bool pv = gq < G && col < NMO;
            const int gg = pv ? gq : 0;
            const int64_t wo = grp * G + gg;
            const bool ok = pv && col < P.n_mo && wo < io.M;
            double g1[2 * NS], g2[2 * NS];
#pragma unroll
            for (int i = 0; i < 2 * NS; ++i) {
              g1[i] = (pv && i < ne) ? sGam[(gg * ne + i) * NMO + col] : 0.0;
              g2[i] = (pv && i < ne) ? sGam2[(gg * ne + i) * NMO + col] : 0.0;
            }
            double racc = 0.0;
            int cur = -1;
            for (int rw = 0; rw < kChunk; ++rw) {
              const int R = chunk * kChunk + rw;
              if (P.ao_orig[R] < 0) continue;
              const double *trow = tile + rw * S;
              double t = 0.0;
#pragma unroll
              for (int i = 0; i < 2 * NS; ++i)
                if (i < ne) t = fma(trow[gg * ne + i], g2[i], fma(trow[GE::opCol(gg * ne + i)], g1[i], t));
              const double cf = ok ? cfr[(((rw >> 2) * NT) + (col >> 3)) * 32 + 4 * (col & 7) + (rw & 3)] : 0.0;
              double a = cf * t;
#pragma unroll
              for (int mm = 1; mm < CW; mm <<= 1) a += shfl_xor_d(a, mm);
              const int at = row_atom[R];
              if (at != cur) {  // the same lane owns walker gg in every chunk and pass: ordered read-modify-writes
                if (cur >= 0 && pv && col == 0 && wo < io.M) dEo[(wo * P.n_atoms + cur) * 3 + cmp] += racc;
                cur = at;
                racc = 0.0;
              }
              racc += a;
            }
            if (cur >= 0 && pv && col == 0 && wo < io.M) dEo[(wo * P.n_atoms + cur) * 3 + cmp] += racc;
          }
          __syncwarp();
          ++chunk;
        }
      }
      __syncwarp();
    }
  }
}

#ifndef QMC_VARIANT_TU  // (the per-variant translation units hold only the template kernels)
// d (V_en + V_nn) / d R_alpha (eq. 1): -Z_alpha sum_i (r_i - R_alpha) / |r_i - R_alpha|^3
// - Z_alpha sum_beta Z_beta (R_alpha - R_beta) / |R_alpha - R_beta|^3.  One thread per walker; writes every entry of dE.
__global__ void __launch_bounds__(128)
    nuclear_potential_gradient_kernel(const __grid_constant__ SysParams P, const double *__restrict__ rin, const int64_t M,
                                      double *__restrict__ dE) {
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= M) return;
  for (int a = 0; a < P.n_atoms; ++a) {
    const double Xa = P.atom[a][0], Ya = P.atom[a][1], Za = P.atom[a][2], Q = P.atom[a][3];
    double gx = 0.0, gy = 0.0, gz = 0.0;
    for (int b = 0; b < P.n_atoms; ++b) {
      if (b == a) continue;
      const double dx = Xa - P.atom[b][0], dy = Ya - P.atom[b][1], dz = Za - P.atom[b][2];
      const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
      const double s = -Q * P.atom[b][3] / (r2 * sqrt(r2));
      gx = fma(s, dx, gx);
      gy = fma(s, dy, gy);
      gz = fma(s, dz, gz);
    }
    for (int i = 0; i < P.n_e; ++i) {
      const double dx = rin[((int64_t)i * 3 + 0) * M + w] - Xa, dy = rin[((int64_t)i * 3 + 1) * M + w] - Ya,
                   dz = rin[((int64_t)i * 3 + 2) * M + w] - Za;
      const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
      const double s = -Q / (r2 * sqrt(r2));
      gx = fma(s, dx, gx);
      gy = fma(s, dy, gy);
      gz = fma(s, dz, gz);
    }
    double *o = dE + (w * P.n_atoms + a) * 3;
    o[0] = gx;
    o[1] = gy;
    o[2] = gz;
  }
}

// Force estimator, eq. 7 (reading Q23): per column j of [M][3 n_atoms]
//   term1_j = -(1/M) sum_m dE[m][j],   term2_j = -(2/M) sum_m (E_L[m] - E_v) dlnpsi[m][j].
// Block b sums a contiguous range of rows (Kahan), one block per column finishes in a fixed order.  stats[0] = E_v.
__global__ void __launch_bounds__(128) force_partial_kernel(const double *__restrict__ eloc, const double *__restrict__ dE,
                                                            const double *__restrict__ dl, int64_t M, int nc,
                                                            const double *__restrict__ stats, double *__restrict__ partial) {
  const double ev = stats[0];
  const int64_t rows = (M + gridDim.x - 1) / gridDim.x;
  const int64_t m0 = (int64_t)blockIdx.x * rows, m1 = (m0 + rows < M) ? m0 + rows : M;
  for (int j = threadIdx.x; j < nc; j += blockDim.x) {
    double s1 = 0.0, c1 = 0.0, s2 = 0.0, c2 = 0.0;
    for (int64_t m = m0; m < m1; ++m) {
      double yv = dE[m * nc + j] - c1, t = s1 + yv;
      c1 = (t - s1) - yv;
      s1 = t;
      yv = (eloc[m] - ev) * dl[m * nc + j] - c2;
      t = s2 + yv;
      c2 = (t - s2) - yv;
      s2 = t;
    }
    partial[((int64_t)blockIdx.x * 2 + 0) * nc + j] = s1;
    partial[((int64_t)blockIdx.x * 2 + 1) * nc + j] = s2;
  }
}
__global__ void __launch_bounds__(128) force_final_kernel(const double *__restrict__ partial, int nblk, int nc, int64_t M,
                                                          const double *__restrict__ stats, double *__restrict__ res) {
  // block (j, which): thread t adds the block partials t, t + 128, ... in order, then a fixed tree
  __shared__ double sh[128];
  const int j = blockIdx.x % nc, which = blockIdx.x / nc;
  double s = 0.0, c = 0.0;
  for (int b = threadIdx.x; b < nblk; b += blockDim.x) {
    const double yv = partial[((int64_t)b * 2 + which) * nc + j] - c, t = s + yv;
    c = (t - s) - yv;
    s = t;
  }
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int w = 64; w > 0; w >>= 1) {
    if ((int)threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) {  // res (mapped host memory) = {E_v, stderr, term1[nc], term2[nc]}
    res[2 + which * nc + j] = (which == 0 ? -1.0 : -2.0) * sh[0] / (double)M;
    if (blockIdx.x == 0) { res[0] = stats[0]; res[1] = stats[1]; }
  }
}

#endif  // QMC_VARIANT_TU
// ---------------------------------------------------------------------------------
// Persistent all-electron Metropolis (readings Q9, Q10).
// Walker coordinates and log|Psi| stay in registers for all sweeps.
// ---------------------------------------------------------------------------------
template <int NS, int NMO, bool X, int WPB, bool EEN = false, bool BF = false>
__global__ void __launch_bounds__(WPB * 32, QMC_MINBLOCKS)
    metropolis_kernel(const __grid_constant__ SysParams P, const WalkerIO io, const MetroParams mp) {
  extern __shared__ __align__(16) unsigned char smem[];
  const double *sC;
  const double *sExp;
  const DetRec *sDet;
  double *wsBase;
  load_constants<NMO>(P, smem, sC, sExp, sDet, wsBase);
  using GE = Geo<NS, NMO>;
  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0), lane = threadIdx.x & 31;  // shfl: tells the compiler it is warp-uniform
  // per-warp scratch: the evaluator's, then the draws of TWO sweeps (they survive the evaluation in between):
  // G (ceil(3 n_e / 2) + 1) Philox blocks per sweep rarely fill the 32 lanes evenly (CO: 44 = 32 + 12), two sweeps' worth
  // do better (88 of 96)
  constexpr int DR = kDrawDoubles<NS>;  // one sweep: normals [G][3 n_e] (<= 96 doubles), then log u [G]
  double *ws = wsBase + warp * (GE::totalC(true) + 2 * DR);
  const double2 *sLogT = reinterpret_cast<const double2 *>(sExp + kExpTab);  // log_pos table
  const double2 *sSinT = sLogT + 64;                                         // sincos_2pi table
  double *sDraw = ws + GE::totalC(true);
  const double *sRes = ws + GE::oResC(true);
  const int ne = X ? 2 * NS : P.n_e, G = X ? GE::GMAX : P.G, nc = 3 * ne, npair = (nc + 1) / 2;
  const int g = lane / ne, e = lane - g * ne;
  const int64_t n_groups = (io.M + G - 1) / G;
  const int wpb = (int)(blockDim.x >> 5);  // warps launched per block (<= WPB, the launch bound)
  const int64_t stride = (int64_t)gridDim.x * wpb;
  unsigned long long acc_count = 0;
  for (int64_t grp = (int64_t)blockIdx.x * wpb + warp; grp < n_groups; grp += stride) {
    const int64_t w = grp * G + g;
    const bool own = (g < G) && (w < io.M);
    const int rg = (own ? g : 0) * 4;
    double x, y, z;
    if (own) {
      x = io.r_out[((int64_t)e * 3 + 0) * io.M + w];
      y = io.r_out[((int64_t)e * 3 + 1) * io.M + w];
      z = io.r_out[((int64_t)e * 3 + 2) * io.M + w];
    } else {
      dummy_xyz(lane, x, y, z);
    }
    double lp = 0.0, sg = 0.0;
    if (mp.resume && own) {
      lp = io.logpsi[w];
      sg = io.sign[w];
    }
    // sweep -1 evaluates the starting point (always "accepted", no draws) unless a previous launch left it
    for (int sw = mp.resume ? 0 : -1; sw < mp.n_sweeps; ++sw) {
      double xp = x, yp = y, zp = z, logu = 0.0;
      if (sw >= 0) {
        // --- draws: lanes share the (sweep, walker, pair) Philox blocks of the G walkers, two sweeps at a time
        if ((sw & 1) == 0) {
          const int per = G * (npair + 1), nsw = (sw + 1 < mp.n_sweeps) ? 2 : 1;
          for (int idx = lane; idx < nsw * per; idx += 32) {
            const int ds = (idx >= per) ? 1 : 0, id2 = idx - ds * per;
            const int dg = id2 / (npair + 1), j = id2 - dg * (npair + 1);
            const uint64_t gw = (uint64_t)(mp.walker_offset + grp * G + dg);
            uint32_t o[4];
            philox4x32_10((uint32_t)gw, mp.sweep0 + (uint32_t)(sw + ds), (j == npair) ? 0xFFFFFFFFu : (uint32_t)j,
                          (uint32_t)(gw >> 32), mp.key0, mp.key1, o);
            const double lu = log_pos(u53(o[0], o[1]), sLogT, P.mc);
            double *dst = sDraw + ds * DR;
            if (j == npair) {
              dst[96 + dg] = lu;
            } else {
              const double rho = sqrt_pos(-2.0 * lu);
              double sn, cs;
              sincos_2pi(u53(o[2], o[3]), sSinT, P.mc, sn, cs);
              dst[dg * nc + 2 * j] = rho * cs;
              if (2 * j + 1 < nc) dst[dg * nc + 2 * j + 1] = rho * sn;
            }
          }
          __syncwarp();
        }
        const double *sProp = sDraw + (sw & 1) * DR, *sLogU = sProp + 96;
        if (own) {
          xp = fma(mp.step, sProp[g * nc + 3 * e + 0], x);
          yp = fma(mp.step, sProp[g * nc + 3 * e + 1], y);
          zp = fma(mp.step, sProp[g * nc + 3 * e + 2], z);
        }
        logu = sLogU[own ? g : 0];
      }
      eval_walkers<NS, NMO, false, X, false, false, EEN, 0, BF>(P, sExp, sC, sDet, ws, xp, yp, zp, lane);
      const double lp2 = sRes[rg + 0], sg2 = sRes[rg + 1];
      // accept iff log u < 2 (log|Psi'| - log|Psi|): false for NaN and for Psi' = 0
      const bool ok = (sw < 0) || (own && (logu < 2.0 * (lp2 - lp)));
      if (ok) { x = xp; y = yp; z = zp; lp = lp2; sg = sg2; }
      if (sw >= 0 && own && e == 0) {
        if (mp.accept) mp.accept[(int64_t)sw * io.M + w] = ok ? 1 : 0;
        acc_count += ok ? 1 : 0;
      }
      __syncwarp();
    }
    if (own) {
      io.r_out[((int64_t)e * 3 + 0) * io.M + w] = x;
      io.r_out[((int64_t)e * 3 + 1) * io.M + w] = y;
      io.r_out[((int64_t)e * 3 + 2) * io.M + w] = z;
      if (e == 0) {
        if (io.logpsi) io.logpsi[w] = lp;
        if (io.sign) io.sign[w] = sg;
      }
    }
    __syncwarp();
  }
  if (mp.n_accepted) {
    for (int m = 16; m > 0; m >>= 1) acc_count += __shfl_xor_sync(0xffffffffu, acc_count, m);
    if (lane == 0 && acc_count) atomicAdd(mp.n_accepted, acc_count);
  }
}

#ifndef QMC_VARIANT_TU  // (the per-variant translation units hold only the template kernels)
// every group on the explicit kernel's work list (qmc_local_energy_explicit)
__global__ void __launch_bounds__(256) list_all_groups_kernel(int *__restrict__ count, int *__restrict__ list,
                                                              int *__restrict__ done, int n_groups) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_groups; i += gridDim.x * blockDim.x) {
    list[i] = i;
    done[i] = 0;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) *count = n_groups;
}

// acc[i] += x[i]  (E_L on every sweep, BASELINE config 5)
__global__ void __launch_bounds__(256) accumulate_kernel(double *__restrict__ acc, const double *__restrict__ x, int64_t M) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < M; i += (int64_t)gridDim.x * blockDim.x) acc[i] += x[i];
}

// ---------------------------------------------------------------------------------
// Gradient estimator of eq. 6: grad_p = (2/M) sum_m O[m][p] (E_L[m] - E_v).
// Deterministic: block b sums its contiguous rows per column (Kahan), then one thread per column adds
// the block partials in order.  stats[0] = E_v (batch_stats_kernel).
// ---------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) gradient_partial_kernel(const double *__restrict__ eloc, const double *__restrict__ O,
                                                               int64_t M, int np, const double *__restrict__ stats,
                                                               double *__restrict__ partial) {
  const double ev = stats[0];
  const int64_t rows = (M + gridDim.x - 1) / gridDim.x;
  const int64_t m0 = (int64_t)blockIdx.x * rows, m1 = (m0 + rows < M) ? m0 + rows : M;
  for (int p = threadIdx.x; p < np; p += blockDim.x) {
    double s = 0.0, c = 0.0;
    for (int64_t m = m0; m < m1; ++m) {
      const double y = O[m * np + p] * (eloc[m] - ev) - c, t = s + y;
      c = (t - s) - y;
      s = t;
    }
    partial[(int64_t)blockIdx.x * np + p] = s;
  }
}
__global__ void __launch_bounds__(128) gradient_final_kernel(const double *__restrict__ partial, int nblk, int np, int64_t M,
                                                             const double *__restrict__ stats, double *__restrict__ res) {
  // one block per parameter: thread t adds the block partials t, t + 128, ... in order, then a fixed tree
  __shared__ double sh[128];
  const int p = blockIdx.x;
  double s = 0.0, c = 0.0;
  for (int b = threadIdx.x; b < nblk; b += blockDim.x) {
    const double y = partial[(int64_t)b * np + p] - c, t = s + y;
    c = (t - s) - y;
    s = t;
  }
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int w = 64; w > 0; w >>= 1) {
    if ((int)threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) {  // res (mapped host memory) = {E_v, stderr, grad[0 .. np-1]}
    res[2 + p] = 2.0 * sh[0] / (double)M;
    if (p == 0) { res[0] = stats[0]; res[1] = stats[1]; }
  }
}

// ---------------------------------------------------------------------------------
// Fused eq. 6: finish grad_p = (2/M) [sum_w O_p E_L - (sum_w O_p)(sum_w E_L)/M] from the per-warp
// partial sums of local_energy_kernel<..., FUSE> and the parked rows of the groups that took the explicit route
// (their E_L is read back from eloc, where explicit_energy_kernel wrote it).  The work list is filled in a
// non-deterministic order, so order_flagged_kernel ranks its entries by group index first: every sum below then
// runs in a fixed order and the result is bit-repeatable.
// ---------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) order_flagged_kernel(const int *__restrict__ fb_count, const int *__restrict__ fb_list,
                                                             int cap, int *__restrict__ order) {
  const int n = min(*fb_count, cap);
  for (int e = threadIdx.x; e < n; e += blockDim.x) {
    const int g = fb_list[e];
    int rank = 0;
    for (int k = 0; k < n; ++k) rank += (fb_list[k] < g) ? 1 : 0;  // group indices are distinct
    order[rank] = e;
  }
}

__device__ __forceinline__ double block_tree_128(double v, double *sh) {
  sh[threadIdx.x] = v;
  __syncthreads();
  for (int w = 64; w > 0; w >>= 1) {
    if ((int)threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
    __syncthreads();
  }
  const double r = sh[0];
  __syncthreads();
  return r;
}

__global__ void __launch_bounds__(128)
    fused_gradient_final_kernel(const double *__restrict__ part, int n_warps, int np, const int *__restrict__ fb_count,
                                const int *__restrict__ fb_list, const int *__restrict__ order, const double *__restrict__ fbO,
                                int cap, const double *__restrict__ eloc, int G, int64_t M, int nj,
                                const int *__restrict__ det_orig, const int *__restrict__ fb_over, double *__restrict__ res) {
  __shared__ double sh[128];
  const int p = blockIdx.x;
  double so = 0.0, soe = 0.0, se = 0.0;
  for (int b = threadIdx.x; b < n_warps; b += blockDim.x) {  // thread t: warps t, t + 128, ... in order
    so += part[(int64_t)p * n_warps + b];
    soe += part[(int64_t)(np + p) * n_warps + b];
    se += part[(int64_t)2 * np * n_warps + b];
  }
  const int n = fb_count ? min(*fb_count, cap) : 0;
  for (int k = threadIdx.x; k < n; k += blockDim.x) {        // listed groups in order of their group index
    const int e = order[k];
    const int64_t grp = fb_list[e];
    for (int wg = 0; wg < G; ++wg) {
      const int64_t wo = grp * G + wg;
      if (wo < M) {
        const double v = fbO[((int64_t)e * G + wg) * np + p], E = eloc[wo];
        so += v;
        soe = fma(v, E, soe);
        se += E;
      }
    }
  }
  const double SO = block_tree_128(so, sh), SOE = block_tree_128(soe, sh), SE = block_tree_128(se, sh);
  if (threadIdx.x == 0) {  // res (mapped host memory) = {E_v, -, grad[0 .. np-1]}; rows were in kernel order
    const double ev = SE / (double)M;
    res[2 + ((p < nj) ? p : nj + det_orig[p - nj])] = 2.0 * (SOE - SO * ev) / (double)M;
    if (p == 0) { res[0] = ev; res[1] = (double)*fb_over; }  // res[1] != 0: the parking area overflowed
  }
}

// ---------------------------------------------------------------------------------
// batch mean and standard error (eq. 3).  One launch, every SM: block b takes a contiguous range of
// the M values and reduces it to {n_b, mean_b, M2_b = sum (x - mean_b)^2} (two passes over its own range, Kahan
// per thread, fixed shuffle tree); the block that finishes last combines the partials pairwise in a fixed tree
// with the exact update  n = n_a + n_b, d = mean_b - mean_a, mean = mean_a + d n_b / n,
// M2 = M2_a + M2_b + d^2 n_a n_b / n  -- deterministic, no atomics on the data -- and writes
// out[0] = mean, out[1] = stderr (out may be mapped host memory).
// ---------------------------------------------------------------------------------
constexpr int kStatsThreads = 256;
__device__ __forceinline__ double block_sum_256(double v, double *sh) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int m = 16; m > 0; m >>= 1) v += shfl_xor_d(v, m);
  __syncthreads();
  if (lane == 0) sh[warp] = v;
  __syncthreads();
  double t = (threadIdx.x < (kStatsThreads >> 5)) ? sh[threadIdx.x] : 0.0;
  if (warp == 0) {
    for (int m = 4; m > 0; m >>= 1) t += shfl_xor_d(t, m);
    if (lane == 0) sh[8] = t;
  }
  __syncthreads();
  return sh[8];
}

__global__ void __launch_bounds__(kStatsThreads) batch_stats_kernel(const double *__restrict__ x, int64_t M, double *__restrict__ partial,
                                                                    unsigned int *__restrict__ done, double *__restrict__ out) {
  __shared__ double sh[9];
  __shared__ double cn[kStatsThreads], cm[kStatsThreads], c2[kStatsThreads];
  __shared__ int is_last;
  const int64_t per = (M + gridDim.x - 1) / gridDim.x;
  const int64_t i0 = (int64_t)blockIdx.x * per, i1 = (i0 + per < M) ? i0 + per : M;
  const double nb = (i1 > i0) ? (double)(i1 - i0) : 0.0;
  double s = 0.0, c = 0.0;
  for (int64_t i = i0 + threadIdx.x; i < i1; i += kStatsThreads) {
    const double y = x[i] - c, t = s + y;
    c = (t - s) - y;
    s = t;
  }
  const double tot = block_sum_256(s, sh);
  const double mean = (nb > 0.0) ? tot / nb : 0.0;
  s = 0.0;
  c = 0.0;
  for (int64_t i = i0 + threadIdx.x; i < i1; i += kStatsThreads) {
    const double d = x[i] - mean;
    const double y = d * d - c, t = s + y;
    c = (t - s) - y;
    s = t;
  }
  const double m2 = block_sum_256(s, sh);
  if (threadIdx.x == 0) {
    partial[3 * blockIdx.x + 0] = nb;
    partial[3 * blockIdx.x + 1] = mean;
    partial[3 * blockIdx.x + 2] = m2;
    __threadfence();
    is_last = (atomicAdd(done, 1u) == gridDim.x - 1) ? 1 : 0;
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  // thread t folds the partials t, t + 256, ... in order, then a fixed binary tree over the threads
  double n = 0.0, mu = 0.0, q = 0.0;
  for (int b = threadIdx.x; b < (int)gridDim.x; b += kStatsThreads) {
    const double n2 = __ldcg(partial + 3 * b), mu2 = __ldcg(partial + 3 * b + 1), q2 = __ldcg(partial + 3 * b + 2);
    if (n2 > 0.0) {
      const double nt = n + n2, dl = mu2 - mu;
      mu = fma(dl, n2 / nt, mu);
      q = q + q2 + dl * dl * (n * n2 / nt);
      n = nt;
    }
  }
  cn[threadIdx.x] = n; cm[threadIdx.x] = mu; c2[threadIdx.x] = q;
  __syncthreads();
  for (int w = kStatsThreads / 2; w > 0; w >>= 1) {
    if ((int)threadIdx.x < w) {
      const double na = cn[threadIdx.x], nb2 = cn[threadIdx.x + w];
      if (nb2 > 0.0) {
        const double nt = na + nb2, dl = cm[threadIdx.x + w] - cm[threadIdx.x];
        cm[threadIdx.x] = fma(dl, nb2 / nt, cm[threadIdx.x]);
        c2[threadIdx.x] = c2[threadIdx.x] + c2[threadIdx.x + w] + dl * dl * (na * nb2 / nt);
        cn[threadIdx.x] = nt;
      }
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    out[0] = cm[0];
    out[1] = (M > 1) ? sqrt(c2[0] / (double)(M - 1) / (double)M) : 0.0;
    *done = 0u;  // ready for the next launch on this stream
  }
}

// ---------------------------------------------------------------------------------
// FP64 peak microbenchmarks (roofline denominator; BASELINE.json north_star)
// ---------------------------------------------------------------------------------
template <int KIND>
__global__ void __launch_bounds__(256) fp64_peak_kernel(double *out, int iters, double seed) {
  double a[8], m0[4], m1[4];
#pragma unroll
  for (int i = 0; i < 8; ++i) a[i] = seed + threadIdx.x * 1e-3 + i;
#pragma unroll
  for (int i = 0; i < 4; ++i) { m0[i] = 0.0; m1[i] = 0.0; }
  const double x = 1.0 + seed * 1e-9, y = seed * 1e-7;
  for (int it = 0; it < iters; ++it) {
    if (KIND == 0 || KIND == 2) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = fma(a[i], x, y);
    }
    if (KIND == 1 || KIND == 2) {
#pragma unroll
      for (int i = 0; i < 4; ++i) dmma884(m0[i], m1[i], x, y);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += a[i];
#pragma unroll
  for (int i = 0; i < 4; ++i) s += m0[i] + m1[i];
  if (s == 123.456) out[0] = s;  // keep the work alive
}

// Operand-form and latency probes of the FP64 pipe (what DESIGN.md section 6 quotes), 32 DFMA per thread and iteration:
//   KIND 3: a = fma(a, x, a)         two distinct registers per instruction, 16 independent chains
//   KIND 4: a = fma(b, c, a)         three distinct registers per instruction, 8 independent chains
//   KIND 5: a = fma(a, x, y)         ONE dependent chain (launched with one warp per SM sub-partition): latency
template <int KIND>
__global__ void __launch_bounds__(256) fp64_probe_kernel(double *out, int iters, double seed) {
  double s = 0.0;
  const double x = 1.0 + seed * 1e-9, y = seed * 1e-7;
  if (KIND == 3) {
    double a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = seed * 1e-3 + threadIdx.x * 1e-6 + i * 1e-4;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = fma(a[i], x, a[i]);
    }
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
  } else if (KIND == 4) {
    double a[8], b[8], c[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = seed + i; b[i] = 1.0 + (threadIdx.x + i) * 1e-9; c[i] = 1.0 - (threadIdx.x + 2 * i) * 1e-9; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = fma(b[i], c[(i + r) & 7], a[i]);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
  } else {
    double a = seed + threadIdx.x * 1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int r = 0; r < 32; ++r) a = fma(a, x, y);
    }
    s = a;
  }
  if (s == 123.456) out[0] = s;
}

#endif  // QMC_VARIANT_TU
}  // namespace qmc
