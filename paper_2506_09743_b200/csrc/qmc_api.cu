// qmc_api.cu -- host side of libqmcb200: the C ABI of include/qmc.h.
// Setup preprocessing (shell grouping, excitation descriptors relative to determinant 0:
// PAPER.md:325 "A_X is constructed by replacing some columns of A_0"), dispatch to the
// compiled (NS, NMO) instantiations, launch geometry, error reporting.
#include "../../include/qmc.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <mutex>
#include <unordered_map>
#include <vector>

#include "qmc_variant.cuh"

using namespace qmc;

namespace qmc {  // the instantiations, one translation unit each (qmc_variant_*.cu)
Variant variant_1_2();
Variant variant_2_2();
Variant variant_3_8();
Variant variant_7_14();
Variant variant_4_8();
Variant variant_8_16();
}  // namespace qmc

namespace {

thread_local std::string g_cuda_err;
thread_local int64_t g_launches = 0;

int cuda_fail(cudaError_t e, const char *what) {
  g_cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
  return QMC_ECUDA;
}
#define CK(call)                                   \
  do {                                             \
    cudaError_t e__ = (call);                      \
    if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
  } while (0)

const std::vector<Variant> &variants() {
  static const std::vector<Variant> v = {
#ifndef QMC_ONLY_CO  // (experiments: build the headline instantiation only)
      variant_1_2(),   // H2-like
      variant_2_2(),   // LiH-like single determinant
      variant_3_8(),   // Li2-like
#endif
      variant_7_14(),  // CO-like (headline)
#ifndef QMC_ONLY_CO
      variant_4_8(),   // generic, runtime electron counts
      variant_8_16(),  // generic upper bound
#endif
  };
  return v;
}

// Scratch of the handle-less reductions (qmc_batch_stats, qmc_energy_gradient), one per (device, stream), created on
// first use and kept for the life of the process: block partials and the completion counter in device memory, the
// result in mapped page-locked host memory that the last block writes directly (no allocation, no copy on the call).
struct ReduceScratch {
  double *d_partial = nullptr;   // [kReduceBlocks][3] {n, mean, M2} of batch_stats_kernel
  unsigned int *d_done = nullptr;
  double *d_stats = nullptr;     // [2] mean, stderr in device memory (read by the gradient kernels)
  double *h_res = nullptr;       // mapped host memory: [2] mean, stderr, then [res_params] gradient
  double *d_res = nullptr;       // device alias of h_res
  size_t res_params = 0;
  double *d_gpart = nullptr;     // [blocks][n_param] partials of gradient_partial_kernel
  size_t gpart_doubles = 0;
};
constexpr int kBfTablesMinDets = 8;  // backflow E_L: expansions up to this size take the explicit kernel alone
constexpr int kReduceBlocks = 592;  // 4 per SM on 148 SMs; any value gives the same result up to rounding order
std::mutex g_reduce_mu;
std::unordered_map<uint64_t, ReduceScratch> g_reduce;

int device_of(const void *p, int *dev) {
  cudaPointerAttributes at{};
  cudaError_t e = cudaPointerGetAttributes(&at, p);
  if (e != cudaSuccess) return cuda_fail(e, "cudaPointerGetAttributes");
  if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) {
    g_cuda_err = "pointer is not device memory";
    return QMC_ECUDA;
  }
  *dev = at.device;
  return QMC_OK;
}

// the scratch of (dev, st) with room for n_param gradient entries and gpart doubles of partials
int reduce_scratch(int dev, cudaStream_t st, size_t n_param, size_t gpart, ReduceScratch **out) {
  std::lock_guard<std::mutex> lock(g_reduce_mu);
  ReduceScratch &r = g_reduce[((uint64_t)(uint32_t)dev << 48) ^ (uint64_t)(uintptr_t)st];
  if (!r.d_partial) {
    CK(cudaMalloc(&r.d_partial, sizeof(double) * 3 * kReduceBlocks));
    CK(cudaMalloc(&r.d_done, sizeof(unsigned int)));
    CK(cudaMemset(r.d_done, 0, sizeof(unsigned int)));
    CK(cudaMalloc(&r.d_stats, sizeof(double) * 2));
  }
  if (!r.h_res || r.res_params < n_param) {  // grow (previous results have been consumed: the calls synchronise)
    if (r.h_res) {
      CK(cudaStreamSynchronize(st));
      cudaFreeHost(r.h_res);
      r.h_res = nullptr;
    }
    const size_t np = std::max<size_t>(n_param, 1024);
    CK(cudaHostAlloc(&r.h_res, sizeof(double) * (2 + np), cudaHostAllocMapped));
    CK(cudaHostGetDevicePointer(&r.d_res, r.h_res, 0));
    r.res_params = np;
  }
  if (r.gpart_doubles < gpart) {
    if (r.d_gpart) {
      CK(cudaStreamSynchronize(st));
      cudaFree(r.d_gpart);
      r.d_gpart = nullptr;
    }
    CK(cudaMalloc(&r.d_gpart, sizeof(double) * gpart));
    r.gpart_doubles = gpart;
  }
  *out = &r;
  return QMC_OK;
}

// ---- qmc_batch_stats_static: the allocation-free entry point.  Its scratch (block partials {n, mean, M2} of
// batch_stats_kernel, then the completion counter) is this file-scope device array: every GPU that loads the library
// holds these kStaticScratchBytes until the process exits.  In host code the array's NAME is a host-side stand-in, not
// a device address; the address comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr int kStaticBlocks = 256;                                   // blocks of the launch = partials held
constexpr int64_t kStaticMaxM = (int64_t)1 << 26;                    // 67 108 864 values (512 MiB of doubles)
constexpr size_t kStaticPartialBytes = sizeof(double) * 3 * kStaticBlocks;
constexpr size_t kStaticScratchBytes = kStaticPartialBytes + 256;    // + the counter, on its own 256-byte line
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
unsigned char *g_static_ptr[kStaticMaxDevices] = {};                 // device address of g_static_scratch, per device

double sto_norm(int n, int l, int m, double zeta) {
  double fact = 1.0;
  for (int i = 2; i <= 2 * n; ++i) fact *= i;
  const double radial = std::pow(2.0 * zeta, n + 0.5) / std::sqrt(fact);
  const double pi = 3.14159265358979323846;
  double ang = 1.0 / (2.0 * std::sqrt(pi));
  if (l == 1) ang = std::sqrt(3.0 / (4.0 * pi));
  if (l == 2) ang = (m <= 2) ? 0.5 * std::sqrt(15.0 / pi) : ((m == 3) ? 0.25 * std::sqrt(15.0 / pi) : 0.25 * std::sqrt(5.0 / pi));
  return radial * ang;
}

}  // namespace

struct qmc_system {
  int device = 0;
  SysParams P{};
  Variant var{};
  int smem_el = 0, smem_psi = 0;  // dynamic shared memory of the E_L kernels (kWarpsEl warps) / values-only kernels
  int smem_metro = 0;             // ... of the sampler
  int warps_psi = 0, warps_metro = 0;  // warps per block the values-only kernels are launched with
  int blocks_el = 0, blocks_psi = 0, blocks_metro = 0, blocks_expl = 0, blocks_deriv = 0;
  void *d_C = nullptr, *d_dets = nullptr, *d_gen = nullptr, *d_cols = nullptr, *d_orig = nullptr, *d_yrec = nullptr, *d_ytgt = nullptr, *d_rowao = nullptr,
       *d_rownrm = nullptr;
  int n_sm = 0;
  double flops_el = 0, flops_step = 0;
  // scratch of the explicit fallback, one buffer per calling stream (grown on demand, kept until qmc_destroy):
  // no allocation on the hot call, and the call can be captured in a CUDA graph after one warm-up call
  // A buffer that has to grow is retired, not freed (a CUDA graph captured earlier may still replay into it); the
  // accept counter of qmc_metropolis is per stream too.
  struct Scratch {
    void *p = nullptr; size_t bytes = 0; unsigned long long *counter = nullptr;
    void *fuse = nullptr; size_t fuse_bytes = 0;  // qmc_local_energy_gradient: warp partials, parked O rows, order list
    void *bf = nullptr; size_t bf_bytes = 0;      // backflow table route: E vectors per resident warp, flagged-walker list
    int *work = nullptr;                          // {work counter, list counter} of the kernels that deal their groups dynamically
    void *orb = nullptr; size_t orb_bytes = 0;    // orbital_explicit_kernel: partial Gamma per work item, group list, slice counters
  };
  std::mutex scratch_mu;
  std::unordered_map<cudaStream_t, Scratch> scratch;
  std::vector<void *> retired;
  // qmc_local_energy_host: two internal streams and double-buffered device scratch (grown on demand)
  bool fuse_ready = false; // fused E_L + eq. 6 kernel configured (lazily)
  int blocks_fuse = 0, smem_fuse = 0;
  bool bf_ready = false;   // backflow E_L kernels configured (lazily)
  int blocks_bf = 0, blocks_bf_tab = 0, warps_bf_tab = 0, warps_bf = 0;
  void *d_bfdets = nullptr;  // BfDet records of the table route (null: the expansion has general determinants)
  int n_bfdets = 0;
  BfClasses bf_cls{};      // class boundaries of the sorted records
  bool frc_ready = false;  // nuclear energy-gradient kernel configured (lazily)
  int frc_warps = 0, blocks_frc = 0;
  bool orb_ready = false;  // orbital-derivative kernel configured (lazily: most users never call it)
  int orb_warps = 0;
  bool time_kernels = false;  // qmc_set_kernel_timing: events around the two kernels of an E_L call
  cudaEvent_t tev[3] = {nullptr, nullptr, nullptr};
  bool tev_fallback = false;
  int blocks_orb = 0;
  cudaStream_t hst[2] = {nullptr, nullptr};
  double *hbuf[2] = {nullptr, nullptr};
  int64_t hbuf_walkers = 0;
  double *helo = nullptr;  // qmc_vmc_step_host: E_L of the whole batch [helo_walkers]
  int64_t helo_walkers = 0;
};

extern "C" {

const char *qmc_status_string(int status) {
  switch (status) {
    case QMC_OK: return "ok";
    case QMC_EINVAL: return "invalid argument";
    case QMC_EUNSUPPORTED: return "problem outside the compiled limits";
    case QMC_ENOMEM: return "host allocation failed";
    case QMC_ETOOLARGE: return "size beyond the fixed scratch of the allocation-free entry point (qmc_batch_stats_static: M <= 67108864)";
    case QMC_ECUDA: return g_cuda_err.empty() ? "CUDA error" : g_cuda_err.c_str();
    default: return "unknown status";
  }
}

int64_t qmc_launch_count(int reset) {
  int64_t v = g_launches;
  if (reset) g_launches = 0;
  return v;
}

void qmc_destroy(qmc_system_t *s) {
  if (!s) return;
  cudaSetDevice(s->device);
  cudaFree(s->d_C);
  cudaFree(s->d_dets);
  cudaFree(s->d_gen);
  cudaFree(s->d_cols);
  for (cudaEvent_t e : s->tev)
    if (e) cudaEventDestroy(e);
  cudaFree(s->d_orig);
  cudaFree(s->d_yrec);
  cudaFree(s->d_ytgt);
  cudaFree(s->d_rowao);
  cudaFree(s->d_rownrm);
  for (auto &kv : s->scratch) {
    cudaFree(kv.second.p);
    cudaFree(kv.second.counter);
    cudaFree(kv.second.work);
    cudaFree(kv.second.orb);
    cudaFree(kv.second.fuse);
    cudaFree(kv.second.bf);
  }
  for (void *q : s->retired) cudaFree(q);
  for (int i = 0; i < 2; ++i) {
    if (s->hst[i]) cudaStreamDestroy(s->hst[i]);
    cudaFree(s->hbuf[i]);
  }
  cudaFree(s->helo);
  cudaFree(s->d_bfdets);
  delete s;
}

int qmc_setup(const qmc_system_desc_t *d, int device, qmc_system_t **out) {
  if (!d || !out) return QMC_EINVAL;
  *out = nullptr;
  if (d->n_atoms < 1 || !d->atom_xyz || !d->atom_Z) return QMC_EINVAL;
  if (d->n_up < 0 || d->n_dn < 0 || d->n_up + d->n_dn < 1) return QMC_EINVAL;
  if (d->n_ao < 1 || !d->ao_atom || !d->ao_n || !d->ao_l || !d->ao_m || !d->ao_zeta) return QMC_EINVAL;
  if (d->n_mo < 1 || !d->mo_coeff) return QMC_EINVAL;
  if (d->n_det < 1 || !d->ci_coeff) return QMC_EINVAL;
  if ((d->n_up > 0 && !d->det_up) || (d->n_dn > 0 && !d->det_dn)) return QMC_EINVAL;
  for (int b = 0; b < d->n_ao; ++b) {
    const int n = d->ao_n[b], l = d->ao_l[b], m = d->ao_m[b];
    if (n < 1 || n > 4 || l < 0 || l > 2 || l >= n || m < 0 || m > 2 * l) return QMC_EINVAL;
    if (!(d->ao_zeta[b] > 0.0)) return QMC_EINVAL;
    if (d->ao_atom[b] < 0 || d->ao_atom[b] >= d->n_atoms) return QMC_EINVAL;
  }
  const int nsp[2] = {d->n_up, d->n_dn};
  const int32_t *lists[2] = {d->det_up, d->det_dn};
  for (int sp = 0; sp < 2; ++sp)
    for (int n = 0; n < d->n_det; ++n)
      for (int j = 0; j < nsp[sp]; ++j) {
        const int c = lists[sp][(size_t)n * nsp[sp] + j];
        if (c < 0 || c >= d->n_mo) return QMC_EINVAL;
        for (int j2 = 0; j2 < j; ++j2)
          if (lists[sp][(size_t)n * nsp[sp] + j2] == c) return QMC_EINVAL;
      }
  if (d->n_atoms > kMaxAtoms || d->n_up > kMaxSpin || d->n_dn > kMaxSpin || d->n_ao > 256) return QMC_EUNSUPPORTED;

  qmc_system *s = new (std::nothrow) qmc_system;
  if (!s) return QMC_ENOMEM;
  s->device = device;
  SysParams &P = s->P;
  {  // constants of the device's elementary functions (qmc_device.cuh)
    MathConsts &K = P.mc;
    K.e_scale = 92.33248261689366;
    K.e_ln2hi = -6.93147180369123816490e-01 / 64;
    K.e_ln2lo = -1.90821492927058770002e-10 / 64;
    K.e_c5 = 1.0 / 120; K.e_c4 = 1.0 / 24; K.e_c3 = 1.0 / 6;
    K.l_c7 = 1.0 / 7; K.l_c6 = -1.0 / 6; K.l_c5 = 1.0 / 5; K.l_c3 = 1.0 / 3;
    K.l_ln2hi = 6.93147180369123816490e-01; K.l_ln2lo = 1.90821492927058770002e-10;
    K.s_2pi = 6.283185307179586;
    K.s_c7 = -1.0 / 5040; K.s_c5 = 1.0 / 120; K.s_c3 = -1.0 / 6;
    K.s_c8 = 1.0 / 40320; K.s_c6 = -1.0 / 720; K.s_c4 = 1.0 / 24;
  }
  P.n_atoms = d->n_atoms;
  P.n_up = d->n_up;
  P.n_dn = d->n_dn;
  P.n_e = d->n_up + d->n_dn;
  P.n_det = d->n_det;
  P.a_par = d->jastrow_a_par;
  P.a_anti = d->jastrow_a_anti;
  P.b = d->jastrow_b;
  P.en_w0 = d->jastrow_en_w0;
  P.en_w1 = d->jastrow_en_w1;
  P.en_w2 = d->jastrow_en_w2;
  P.has_en = (d->jastrow_en_w0 != 0.0 || d->jastrow_en_w1 != 0.0) ? 1 : 0;
  P.bf_w = d->backflow_w;
  if (!(d->backflow_w == d->backflow_w)) {  // NaN
    delete s;
    return QMC_EINVAL;
  }
  if (d->n_een < 0 || (d->n_een > 0 && !d->een_params)) {
    delete s;
    return QMC_EINVAL;
  }
  if (d->n_een > kMaxEen) {
    delete s;
    return QMC_EUNSUPPORTED;
  }
  P.n_een = d->n_een;
  // D.3 enters eq. 5 once per pair, symmetrised (reading Q22): the kernels run over ordered
  // pairs, so they carry c / 2
  for (int mu = 0; mu < d->n_een; ++mu)
    for (int t = 0; t < 7; ++t) P.een[mu][t] = (t == 0 ? 0.5 : 1.0) * d->een_params[7 * mu + t];
  for (int a = 0; a < d->n_atoms; ++a) {
    for (int c = 0; c < 3; ++c) P.atom[a][c] = d->atom_xyz[3 * a + c];
    P.atom[a][3] = d->atom_Z[a];
  }
  // nuclear repulsion, last term of eq. 1
  P.vnn = 0.0;
  for (int a = 0; a < d->n_atoms; ++a)
    for (int b = a + 1; b < d->n_atoms; ++b) {
      const double dx = P.atom[a][0] - P.atom[b][0], dy = P.atom[a][1] - P.atom[b][1], dz = P.atom[a][2] - P.atom[b][2];
      P.vnn += P.atom[a][3] * P.atom[b][3] / std::sqrt(dx * dx + dy * dy + dz * dz);
    }

  // ---- orbitals actually referenced; excitation descriptors relative to determinant 0
  std::vector<int> used;  // kernel column -> caller MO index
  auto col_of = [&](int mo) {
    for (size_t i = 0; i < used.size(); ++i)
      if (used[i] == mo) return (int)i;
    used.push_back(mo);
    return (int)used.size() - 1;
  };
  std::vector<int> virt[2];  // caller MO index of virtual q
  struct Exc { int k[2]; int p[2][kMaxSpin]; int q[2][kMaxSpin]; double d; int orig; };
  std::vector<Exc> excs(d->n_det);
  bool unsupported = false;
  for (int sp = 0; sp < 2; ++sp)
    for (int j = 0; j < nsp[sp]; ++j) P.ref_col[sp][j] = (int8_t)col_of(lists[sp][j]);
  for (int n = 0; n < d->n_det; ++n) {
    Exc &x = excs[n];
    x.d = d->ci_coeff[n];
    x.orig = n;
    for (int sp = 0; sp < 2; ++sp) {
      int k = 0;
      for (int j = 0; j < nsp[sp]; ++j) {
        const int mo = lists[sp][(size_t)n * nsp[sp] + j];
        if (mo == lists[sp][j]) continue;
        int q = -1;
        for (size_t t = 0; t < virt[sp].size(); ++t)
          if (virt[sp][t] == mo) q = (int)t;
        if (q < 0) {
          virt[sp].push_back(mo);
          q = (int)virt[sp].size() - 1;
        }
        x.p[sp][k] = j;
        x.q[sp][k] = q;
        ++k;
      }
      x.k[sp] = k;
    }
  }
  // Determinant classes (the lanes of a warp take consecutive determinants of one class and run the same code):
  //   0  equal to the reference                      -> their coefficients are summed into P.d_ref
  //   1  one substitution in one spin                 -> one table entry
  //   2  one substitution in each spin                -> two table entries
  //   3  two substitutions in one spin, none in the other -> one 2x2 sub-determinant
  //   4  anything else with at most two per spin      -> two 2x2 sub-determinants (padded with constant entries)
  //   5  more than two substitutions in a spin        -> general sub-determinants (GenDet)
  auto det_class = [](const Exc &x) {
    const int lo = std::min(x.k[0], x.k[1]), hi = std::max(x.k[0], x.k[1]);
    if (hi > 2) return 5;
    if (hi == 0) return 0;
    if (hi == 1) return lo == 0 ? 1 : 2;
    return lo == 0 ? 3 : 4;
  };
  std::stable_sort(excs.begin(), excs.end(), [&](const Exc &a, const Exc &b) { return det_class(a) < det_class(b); });
  int n_cls[6] = {0, 0, 0, 0, 0, 0};
  for (const Exc &x : excs) ++n_cls[det_class(x)];
  const int n_ref = n_cls[0];
  const int n_packed = n_cls[1] + n_cls[2] + n_cls[3] + n_cls[4];  // packed 16-byte records (classes 1-4)
  P.d_ref = 0.0;
  for (int n = 0; n < n_ref; ++n) P.d_ref += excs[n].d;
  P.n_ref = n_ref;
  std::vector<int> det_orig(d->n_det);  // kernel order -> caller's determinant index (parameter derivatives)
  for (int n = 0; n < d->n_det; ++n) det_orig[n] = excs[n].orig;
  P.n_a1 = n_cls[1];
  P.n_a2 = P.n_a1 + n_cls[2];
  P.n_b = P.n_a2 + n_cls[3];
  for (int sp = 0; sp < 2; ++sp) {
    if ((int)virt[sp].size() > kMaxVirt) unsupported = true;
    P.nv[sp] = (int)virt[sp].size();
    if (!unsupported)
      for (int q = 0; q < P.nv[sp]; ++q) P.virt_col[sp][q] = (int8_t)col_of(virt[sp][q]);
  }
  if (unsupported || used.size() > 16) {
    delete s;
    return QMC_EUNSUPPORTED;
  }
  P.n_mo = (int)used.size();
  // column lists of every determinant in kernel MO order (explicit fallback path)
  std::vector<DetCols> cols(d->n_det);
  for (int n = 0; n < d->n_det; ++n) {
    cols[n].d = d->ci_coeff[n];
    for (int sp = 0; sp < 2; ++sp)
      for (int j = 0; j < kMaxSpin; ++j)
        cols[n].col[sp][j] = (j < nsp[sp]) ? (int8_t)col_of(lists[sp][(size_t)n * nsp[sp] + j]) : 0;
  }
  P.n_det_all = d->n_det;

  // ---- pick the instantiation
  const int ns_max = std::max(d->n_up, d->n_dn), nv_max = std::max(P.nv[0], P.nv[1]);
  const Variant *var = nullptr;
  for (const Variant &v : variants())
    if (v.NS >= ns_max && v.NMO >= P.n_mo && v.LP >= nv_max && v.LP >= ns_max &&
        (!v.exact || (d->n_up == v.NS && d->n_dn == v.NS))) {
      var = &v;
      break;
    }
  if (!var) {
    delete s;
    return QMC_EUNSUPPORTED;
  }
  s->var = *var;
  if (P.bf_w != 0.0) {  // the values-only instantiations that evaluate the orbitals at the backflow coordinates
    s->var.k_psi = var->b_psi;
    s->var.k_metro = var->b_metro;
    s->var.k_orb = var->k_orb_b;  // and the orbital-parameter / nuclear log-gradient kernels with the AOs there
    s->var.k_orb_small = var->k_orb_small_b;
    s->var.k_nuc = var->k_nuc_b;
    s->var.k_nuc_small = var->k_nuc_small_b;
    s->var.x_orb = var->x_orb_b;
    s->var.x_orb_small = var->x_orb_small_b;
    s->var.x_nuc = var->x_nuc_b;
    s->var.x_nuc_small = var->x_nuc_small_b;
  }
  if (P.n_een > 0) {  // the instantiations that carry the e-e-n Jastrow kernel
    s->var.k_el = var->e_el;
    s->var.k_psi = var->e_psi;
    s->var.k_metro = var->e_metro;
    s->var.k_expl = var->e_expl;
    s->var.k_el_deriv = var->e_el_deriv;
    if (P.bf_w != 0.0) {  // both: the values-only kernels with D.3 at r and the orbitals at the backflow coordinates
      s->var.k_psi = var->be_psi;
      s->var.k_metro = var->be_metro;
    }
  }
  const int NMO = var->NMO;
  std::vector<DetRec> dets(n_packed);
  std::vector<YRec> yrec;
  std::vector<int2> ytgt;
  std::vector<GenDet> gens;
  for (int n = n_ref + n_packed; n < d->n_det; ++n) {
    GenDet g{};
    g.d = excs[n].d;
    for (int sp = 0; sp < 2; ++sp) {
      g.s[sp].k = (uint8_t)excs[n].k[sp];
      for (int t = 0; t < excs[n].k[sp]; ++t) {
        g.s[sp].p[t] = (uint8_t)excs[n].p[sp][t];
        g.s[sp].q[t] = (uint8_t)excs[n].q[sp][t];
      }
    }
    gens.push_back(g);
  }
  P.n_det = n_packed;
  P.n_gen = (int)gens.size();
  {
    const int LPv = var->LP + 1, TSv = var->NS * LPv + 2;       // Geo::RS (table row stride), Geo::TS (stride per (walker, spin))
    const uint32_t one = (uint32_t)(var->NS * LPv), zero = one + 1;  // constant table entries {1,0}, {0,0}
    // byte offset (for 8-byte entries; the E_L tables hold 16-byte {T, M} entries and double it) of entry
    // (p, q) of spin sp relative to the walker's up-spin table
    auto off8 = [&](int sp, int p, int q) { return (uint32_t)(8 * (sp * TSv + p * LPv + q)); };
    for (int n = 0; n < n_packed; ++n) {
      const Exc &x = excs[n_ref + n];
      const int cls = det_class(x);
      DetRec &r = dets[n];
      r.d = x.d;
      if (cls == 1) {
        const int sp = x.k[0] ? 0 : 1;
        r.up = off8(sp, x.p[sp][0], x.q[sp][0]);
        r.dn = 0;
      } else if (cls == 2) {
        r.up = off8(0, x.p[0][0], x.q[0][0]);
        r.dn = off8(1, x.p[1][0], x.q[1][0]);
      } else if (cls == 3) {
        const int sp = x.k[0] ? 0 : 1;
        r.up = off8(sp, x.p[sp][0], x.q[sp][0]) | (off8(sp, x.p[sp][0], x.q[sp][1]) << 16);  // 11, 12
        r.dn = off8(sp, x.p[sp][1], x.q[sp][0]) | (off8(sp, x.p[sp][1], x.q[sp][1]) << 16);  // 21, 22
      } else {
        uint32_t code[2];
        for (int sp = 0; sp < 2; ++sp) {
          uint32_t i11 = one, i12 = zero, i21 = zero, i22 = one;
          if (x.k[sp] >= 1) i11 = (uint32_t)(x.p[sp][0] * LPv + x.q[sp][0]);
          if (x.k[sp] == 2) {
            i12 = (uint32_t)(x.p[sp][0] * LPv + x.q[sp][1]);
            i21 = (uint32_t)(x.p[sp][1] * LPv + x.q[sp][0]);
            i22 = (uint32_t)(x.p[sp][1] * LPv + x.q[sp][1]);
          }
          code[sp] = i11 | (i12 << 8) | (i21 << 16) | (i22 << 24);
        }
        r.up = code[0];
        r.dn = code[1];
      }
    }
    // Gather lists for Y = d(Sigma/D_0)/dT (orbital-parameter derivatives): per table entry (spin, p, q) the
    // determinants that contain it, as {d_n * cofactor sign, the other spin's sub-determinant code, the cofactor's
    // table index}; entries sorted by list length so that dealing them to lanes round-robin balances the work.
    std::vector<std::vector<YRec>> lists_y((size_t)2 * TSv);
    for (int n = 0; n < n_packed; ++n) {
      const Exc &x = excs[n_ref + n];
      uint32_t code[2];
      for (int sp = 0; sp < 2; ++sp) {
        uint32_t i11 = one, i12 = zero, i21 = zero, i22 = one;
        if (x.k[sp] >= 1) i11 = (uint32_t)(x.p[sp][0] * LPv + x.q[sp][0]);
        if (x.k[sp] == 2) {
          i12 = (uint32_t)(x.p[sp][0] * LPv + x.q[sp][1]);
          i21 = (uint32_t)(x.p[sp][1] * LPv + x.q[sp][0]);
          i22 = (uint32_t)(x.p[sp][1] * LPv + x.q[sp][1]);
        }
        code[sp] = i11 | (i12 << 8) | (i21 << 16) | (i22 << 24);
      }
      for (int sp = 0; sp < 2; ++sp) {
        auto add = [&](int p, int q, double w, uint32_t cof) {
          YRec y{};
          y.w = w;
          y.oth = code[1 - sp];
          y.cof = (uint16_t)cof;
          lists_y[(size_t)sp * TSv + p * LPv + q].push_back(y);
        };
        if (x.k[sp] == 1) {
          add(x.p[sp][0], x.q[sp][0], x.d, one);
        } else if (x.k[sp] == 2) {  // cofactors of {T11 T12; T21 T22}
          const int p0 = x.p[sp][0], p1 = x.p[sp][1], q0 = x.q[sp][0], q1 = x.q[sp][1];
          add(p0, q0, x.d, (uint32_t)(p1 * LPv + q1));
          add(p0, q1, -x.d, (uint32_t)(p1 * LPv + q0));
          add(p1, q0, -x.d, (uint32_t)(p0 * LPv + q1));
          add(p1, q1, x.d, (uint32_t)(p0 * LPv + q0));
        }
      }
    }
    std::vector<int> order;
    for (int t = 0; t < 2 * TSv; ++t)
      if (!lists_y[t].empty()) order.push_back(t);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return lists_y[a].size() > lists_y[b].size(); });
    for (int t : order) {
      ytgt.push_back(make_int2(t, (int)yrec.size()));
      yrec.insert(yrec.end(), lists_y[t].begin(), lists_y[t].end());
    }
    P.n_ytgt = (int)order.size();
    ytgt.push_back(make_int2(0, (int)yrec.size()));  // end of the last list
  }
  P.G = std::max(1, std::min(32 / P.n_e, 16 / var->NS));

  // ---- shell grouping: AOs that share a centre, n, l and zeta share one radial factor
  struct Rec { ShellRec r; std::vector<int> aos; int atom; };
  std::vector<Rec> recs;
  for (int b = 0; b < d->n_ao;) {
    const int at = d->ao_atom[b], n = d->ao_n[b], l = d->ao_l[b];
    const double z = d->ao_zeta[b];
    const int nfun = 2 * l + 1;
    bool full = (b + nfun <= d->n_ao);
    for (int t = 0; full && t < nfun; ++t)
      full = d->ao_atom[b + t] == at && d->ao_n[b + t] == n && d->ao_l[b + t] == l && d->ao_zeta[b + t] == z && d->ao_m[b + t] == t;
    Rec rc;
    rc.atom = at;
    const int k = n - 1 - l;
    rc.r.zeta = z;
    rc.r.c1 = 2.0 * z * (k + l + 1);
    rc.r.c2 = (double)(k * (k + 2 * l + 1));
    rc.r.kd = (double)k;
    rc.r.pad = 0;
    rc.r.dlnN = d->ao_norm ? 0.0 : (n + 0.5) / z;
    int kind;
    if (l == 0) { kind = SH_S; rc.aos = {b}; b += 1; }
    else if (full) { kind = (l == 1) ? SH_P : SH_D; for (int t = 0; t < nfun; ++t) rc.aos.push_back(b + t); b += nfun; }
    else { kind = (l == 1) ? SH_P1 : SH_D1; rc.aos = {b}; b += 1; }
    rc.r.meta = kind | (k << 4) | ((l == 0 || full ? 0 : d->ao_m[rc.aos[0]]) << 8);
    recs.push_back(rc);
  }
  // per atom, shells in order of their radial power k (stable): one SH_POW record ahead of each power > 0
  auto rec_k = [](const Rec &a) { return (a.r.meta >> 4) & 3; };
  std::stable_sort(recs.begin(), recs.end(), [&](const Rec &a, const Rec &b) { return a.atom != b.atom ? a.atom < b.atom : rec_k(a) < rec_k(b); });
  size_t n_pow = 0;
  for (size_t q = 0; q < recs.size(); ++q)
    if (rec_k(recs[q]) > 0 && (q == 0 || recs[q - 1].atom != recs[q].atom || rec_k(recs[q - 1]) != rec_k(recs[q]))) ++n_pow;
  if (recs.size() + (size_t)d->n_atoms + n_pow > (size_t)kMaxShells) {
    delete s;
    return QMC_EUNSUPPORTED;
  }
  // AO rows are laid out in chunks of kChunk (one DMMA pass each); a record never straddles a chunk.
  // The last record of a chunk carries the number of rows the chunk uses (meta >> 20).
  std::vector<ShellRec> shells;
  int n_real_shells = 0;
  std::vector<std::vector<double>> crow;  // kernel AO row -> coefficients of the referenced MOs (or empty = pad)
  std::vector<int> row_ao;                // kernel AO row -> caller's AO index (-1 = pad)
  std::vector<double> row_nrm;            // kernel AO row -> normalisation
  {
    int row = 0;
    int n_real = 0;
    auto last_shell = [&]() -> ShellRec & {  // the last shell record (an atom record cannot carry the flush)
      size_t j = shells.size();
      while ((shells[j - 1].meta & 15) == SH_ATOM || (shells[j - 1].meta & 15) == SH_POW) --j;
      return shells[j - 1];
    };
    size_t i = 0;
    for (int a = 0; a < d->n_atoms; ++a) {
      {  // atom record: {zeta, c1, c2, kd} = {X, Y, Z, charge} (also for a centre without basis functions: V_en)
        ShellRec ar{};
        ar.zeta = d->atom_xyz[3 * a + 0];
        ar.c1 = d->atom_xyz[3 * a + 1];
        ar.c2 = d->atom_xyz[3 * a + 2];
        ar.kd = d->atom_Z[a];
        ar.meta = SH_ATOM;
        shells.push_back(ar);
      }
      int cur_k = 0;
      for (; i < recs.size() && recs[i].atom == a; ++i) {
      const int nf = (int)recs[i].aos.size();
      ++n_real;
      if (rec_k(recs[i]) != cur_k) {  // the shells from here on carry r^k
        cur_k = rec_k(recs[i]);
        ShellRec pr{};
        pr.meta = SH_POW | (cur_k << 4);
        shells.push_back(pr);
      }
      if (row % kChunk + nf > kChunk) {
        last_shell().meta |= (row % kChunk) << 20;
        while (row % kChunk) { crow.emplace_back(); row_ao.push_back(-1); row_nrm.push_back(0.0); ++row; }
      }
      recs[i].r.meta |= (row % kChunk) << 12;
      for (int b : recs[i].aos) {
        const double nrm = d->ao_norm ? d->ao_norm[b] : sto_norm(d->ao_n[b], d->ao_l[b], d->ao_m[b], d->ao_zeta[b]);
        std::vector<double> c(P.n_mo);
        for (int mo = 0; mo < P.n_mo; ++mo) c[mo] = nrm * d->mo_coeff[(size_t)b * d->n_mo + used[mo]];
        crow.push_back(c);
        row_ao.push_back(b);
        row_nrm.push_back(nrm);
        ++row;
      }
      shells.push_back(recs[i].r);
      if (row % kChunk == 0) shells.back().meta |= kChunk << 20;
      }
    }
    if (row % kChunk) {
      last_shell().meta |= (row % kChunk) << 20;
      while (row % kChunk) { crow.emplace_back(); row_ao.push_back(-1); row_nrm.push_back(0.0); ++row; }
    }
    n_real_shells = n_real;
  }
  {  // second half of the row table: kernel AO row -> centre (-1 = pad), for qmc_nuclear_log_gradient
    const size_t n_rows = row_ao.size();
    for (size_t R = 0; R < n_rows; ++R) row_ao.push_back(row_ao[R] < 0 ? -1 : d->ao_atom[row_ao[R]]);
  }
  for (size_t i = 0; i < shells.size(); ++i) P.shells[i] = shells[i];
  const int n_chunks = (int)crow.size() / kChunk, NT = (NMO + 7) / 8, KS = kChunk / 4;
  P.n_chunks = n_chunks;
  // B fragments of mma.m8n8k4 (col-major B[k][n] held by lane 4 n + k)
  std::vector<double> C((size_t)n_chunks * KS * NT * 32, 0.0);
  for (int ch = 0; ch < n_chunks; ++ch)
    for (int ks = 0; ks < KS; ++ks)
      for (int t = 0; t < NT; ++t)
        for (int lane = 0; lane < 32; ++lane) {
          const int k = ch * kChunk + 4 * ks + (lane & 3), n = 8 * t + (lane >> 2);
          if (!crow[k].empty() && n < P.n_mo) C[(((size_t)ch * KS + ks) * NT + t) * 32 + lane] = crow[k][n];
        }
  P.n_shell = (int)shells.size();
  P.n_ao = d->n_ao;
  P.c_doubles = (int)C.size();
  for (int j = 0; j < kExpTab; ++j) C.push_back((double)exp2l((long double)j / kExpTab));  // exp_neg's 2^(j/64)
  {  // Box-Muller tables (qmc_device.cuh: log_pos, sincos_2pi)
    for (int j = 0; j < 64; ++j) {  // piece j of [sqrt(1/2), sqrt(2)): high words 0x3fe6a09e + [j, j+1) * 2^14
      const uint64_t lo = ((uint64_t)(0x3fe6a09eu + ((uint32_t)j << 14))) << 32;
      const uint64_t hi = (((uint64_t)(0x3fe6a09eu + ((uint32_t)(j + 1) << 14))) << 32) - 1;
      double mlo, mhi;
      std::memcpy(&mlo, &lo, 8);
      std::memcpy(&mhi, &hi, 8);
      const double inv = (double)(1.0L / (0.5L * ((long double)mlo + (long double)mhi)));
      C.push_back(inv);
      C.push_back((double)(-logl((long double)inv)));
    }
    const long double two_pi = 6.283185307179586476925286766559L;
    for (int j = 0; j < 64; ++j) {
      C.push_back((double)cosl(two_pi * j / 64));
      C.push_back((double)sinl(two_pi * j / 64));
    }
  }

  // ---- model FP64 work per walker
  {
    const double cexp = 40, cdiv = 20, csqrt = 20, clog = 50, csincos = 80;
    const double ne = P.n_e, nat = P.n_atoms, nsh = n_real_shells, nao = P.n_ao, nmo = P.n_mo, nd = d->n_det;
    const double npair = ne * (ne - 1) / 2;
    double lu_el = 0, lu_st = 0;
    for (int sp = 0; sp < 2; ++sp) {
      const double n = nsp[sp], v = P.nv[sp];
      lu_el += 2 * n * n * n + 3 * 2 * n * n * v + 2 * n * n * n + n + n * cdiv;
      lu_st += 2.0 / 3.0 * n * n * n + 2 * n * n * v + n * cdiv;
    }
    s->flops_el = ne * nat * (8 + csqrt + cdiv) + ne * nsh * (8 + cexp) + ne * nao * 21 + 2 * ne * nao * nmo * 2 +
                  npair * (35 + csqrt + 2 * cdiv) + lu_el + 15 * nd + 100;
    if (P.has_en) {  // D.2 per (electron, nucleus): K, K', K'', gradient and Laplacian shares (the distance is reused)
      s->flops_el += ne * nat * (22 + cdiv);
    }
    const double npr = std::ceil(3 * ne / 2);
    s->flops_step = ne * nat * (8 + csqrt + cdiv) + ne * nsh * (2 + cexp) + ne * nao * 3 + 2 * ne * nao * nmo +
                    npair * (12 + csqrt + cdiv) + lu_st + 3 * nd + 3 * ne * 2 + npr * (10 + clog + csqrt + csincos) + clog;
    if (P.has_en) s->flops_step += ne * nat * (5 + cdiv);
    if (P.n_een > 0) {  // D.3 per (nucleus, ordered pair, term): three Pade factors and their products
      s->flops_el += nat * ne * (ne - 1) * P.n_een * (30 + 3 * cdiv);
      s->flops_step += nat * ne * (ne - 1) * P.n_een * (10 + 3 * cdiv);
    }
  }

  // backflow table route: one compact record per determinant (caller order), when no determinant needs more than two
  // substitutions in a spin
  std::vector<BfDet> bfdets;
  BfClasses bf_cls{};
  if (P.bf_w != 0.0 && gens.empty() && d->n_det <= 65535) {  // (the records carry the caller's index in 16 bits)
    std::vector<Exc> by_orig(excs);
    std::sort(by_orig.begin(), by_orig.end(), [](const Exc &a, const Exc &b) { return a.orig < b.orig; });
    for (const Exc &x : by_orig) {
      BfDet r{};
      r.d = x.d;
      for (int sp = 0; sp < 2; ++sp) {
        r.k[sp] = (uint8_t)x.k[sp];
        for (int t = 0; t < x.k[sp] && t < 2; ++t) {
          r.p[sp][t] = (uint8_t)x.p[sp][t];
          r.q[sp][t] = (uint8_t)x.q[sp][t];
        }
      }
      r.orig = (uint16_t)x.orig;
      bfdets.push_back(r);
    }
    // one loop per class (k_up, k_dn) in the kernel: records sorted by class, caller order within a class
    std::stable_sort(bfdets.begin(), bfdets.end(), [](const BfDet &a, const BfDet &b) { return 3 * a.k[0] + a.k[1] < 3 * b.k[0] + b.k[1]; });
    int at = 0;
    for (int c = 0; c < 9; ++c) {
      bf_cls.start[c] = at;
      while (at < (int)bfdets.size() && 3 * bfdets[at].k[0] + bfdets[at].k[1] == c) ++at;
    }
    bf_cls.start[9] = at;
  }
  // ---- upload
  cudaError_t e = cudaSetDevice(device);
  if (e != cudaSuccess) { delete s; return cuda_fail(e, "cudaSetDevice"); }
  const size_t szC = C.size() * sizeof(double), szD = dets.size() * sizeof(DetRec);
  if ((e = cudaMalloc(&s->d_C, szC)) != cudaSuccess ||
      (e = cudaMalloc(&s->d_dets, szD)) != cudaSuccess ||
      (e = cudaMemcpy(s->d_C, C.data(), szC, cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMemcpy(s->d_dets, dets.data(), szD, cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMalloc(&s->d_gen, std::max<size_t>(gens.size(), 1) * sizeof(GenDet))) != cudaSuccess ||
      (!gens.empty() && (e = cudaMemcpy(s->d_gen, gens.data(), gens.size() * sizeof(GenDet), cudaMemcpyHostToDevice)) != cudaSuccess) ||
      (e = cudaMalloc(&s->d_cols, cols.size() * sizeof(DetCols))) != cudaSuccess ||
      (e = cudaMemcpy(s->d_cols, cols.data(), cols.size() * sizeof(DetCols), cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMalloc(&s->d_orig, det_orig.size() * sizeof(int))) != cudaSuccess ||
      (e = cudaMemcpy(s->d_orig, det_orig.data(), det_orig.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMalloc(&s->d_yrec, std::max<size_t>(yrec.size(), 1) * sizeof(YRec))) != cudaSuccess ||
      (!yrec.empty() && (e = cudaMemcpy(s->d_yrec, yrec.data(), yrec.size() * sizeof(YRec), cudaMemcpyHostToDevice)) != cudaSuccess) ||
      (e = cudaMalloc(&s->d_ytgt, ytgt.size() * sizeof(int2))) != cudaSuccess ||
      (e = cudaMemcpy(s->d_ytgt, ytgt.data(), ytgt.size() * sizeof(int2), cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMalloc(&s->d_rowao, row_ao.size() * sizeof(int))) != cudaSuccess ||
      (e = cudaMemcpy(s->d_rowao, row_ao.data(), row_ao.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMalloc(&s->d_rownrm, row_nrm.size() * sizeof(double))) != cudaSuccess ||
      (e = cudaMemcpy(s->d_rownrm, row_nrm.data(), row_nrm.size() * sizeof(double), cudaMemcpyHostToDevice)) != cudaSuccess) {
    int rc = cuda_fail(e, "qmc_setup upload");
    qmc_destroy(s);
    return rc;
  }
  if (!bfdets.empty()) {
    if ((e = cudaMalloc(&s->d_bfdets, bfdets.size() * sizeof(BfDet))) != cudaSuccess ||
        (e = cudaMemcpy(s->d_bfdets, bfdets.data(), bfdets.size() * sizeof(BfDet), cudaMemcpyHostToDevice)) != cudaSuccess) {
      int rc = cuda_fail(e, "qmc_setup upload (backflow records)");
      qmc_destroy(s);
      return rc;
    }
    s->n_bfdets = (int)bfdets.size();
    s->bf_cls = bf_cls;
  }
  P.exp_tab = (const double *)s->d_C + P.c_doubles;
  P.rng_tab = P.exp_tab + kExpTab;
  P.C = (const double *)s->d_C;
  P.dets = (const DetRec *)s->d_dets;
  P.gen = (const GenDet *)s->d_gen;
  P.det_cols = (const DetCols *)s->d_cols;
  P.det_orig = (const int *)s->d_orig;
  P.yrec = (const YRec *)s->d_yrec;
  P.ytgt = (const int2 *)s->d_ytgt;
  P.ao_orig = (const int *)s->d_rowao;
  P.ao_nrm = (const double *)s->d_rownrm;
  for (int a = 0; a < 16; ++a) P.mo_orig[a] = a < P.n_mo ? used[a] : 0;
  P.n_mo_all = d->n_mo;
  P.smem_const_bytes = (int)((szC + szD + 15) / 16 * 16);
  s->smem_el = P.smem_const_bytes + kWarpsEl * var->ws_doubles * (int)sizeof(double);
  // values-only kernels: the most warps per block (up to the launch bound) that keep QMC_MINBLOCKS blocks' shared
  // memory on an SM -- a long expansion's constants would otherwise cost a whole block of warps
  int sm_smem = 0;
  cudaDeviceGetAttribute(&sm_smem, cudaDevAttrMaxSharedMemoryPerMultiprocessor, device);
  auto fit_warps = [&](int ws_doubles) {
    int w = var->wpb_psi_max;
    while (w > 4 && QMC_MINBLOCKS * (P.smem_const_bytes + w * ws_doubles * (int)sizeof(double) + 1024) > sm_smem) --w;
    return w;
  };
  s->warps_psi = fit_warps(var->psi_ws_doubles);
  s->warps_metro = fit_warps(var->metro_ws_doubles);
  s->smem_psi = P.smem_const_bytes + s->warps_psi * var->psi_ws_doubles * (int)sizeof(double);
  s->smem_metro = P.smem_const_bytes + s->warps_metro * var->metro_ws_doubles * (int)sizeof(double);

  int dev_smem = 0, n_sm = 0;
  cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device);
  if (std::max(s->smem_el, s->smem_metro) > dev_smem) {
    qmc_destroy(s);
    return QMC_EUNSUPPORTED;
  }
  s->n_sm = n_sm;
  const void *ks[5] = {s->var.k_el, s->var.k_psi, s->var.k_metro, s->var.k_expl, s->var.k_el_deriv};
  int *nb[5] = {&s->blocks_el, &s->blocks_psi, &s->blocks_metro, &s->blocks_expl, &s->blocks_deriv};
  const int kw[5] = {kWarpsEl, s->warps_psi, s->warps_metro, kWarpsEl, kWarpsEl};
  const int ksm[5] = {s->smem_el, s->smem_psi, s->smem_metro, s->smem_el, s->smem_el};
  for (int i = 0; i < 5; ++i) {
    if ((e = cudaFuncSetAttribute(ks[i], cudaFuncAttributeMaxDynamicSharedMemorySize, ksm[i])) != cudaSuccess) {
      int rc = cuda_fail(e, "cudaFuncSetAttribute");
      qmc_destroy(s);
      return rc;
    }
    int per_sm = 0;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ks[i], kw[i] * 32, ksm[i])) != cudaSuccess || per_sm < 1) {
      int rc = (e != cudaSuccess) ? cuda_fail(e, "occupancy") : QMC_EUNSUPPORTED;
      qmc_destroy(s);
      return rc;
    }
    *nb[i] = per_sm * n_sm;
  }
  *out = s;
  return QMC_OK;
}

static int launch_eval(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign, double *d_eloc,
                       void *stream, bool el, double *d_O = nullptr, bool explicit_only = false) {
  if (!s || !d_r || M <= 0) return QMC_EINVAL;
  CK(cudaSetDevice(s->device));
  cudaStream_t st = (cudaStream_t)stream;
  WalkerIO io{};
  io.r_in = d_r;
  io.logpsi = d_logpsi;
  io.sign = d_sign;
  io.eloc = d_eloc;
  io.O = d_O;
  io.M = M;
  if (s->P.bf_w != 0.0 && el) {
    // backflow wavefunction: E_L by its own kernels (qmc_backflow.cuh); with d_O their instantiations
    // that also write the parameter derivatives, [M][qmc_n_param] with the backflow weight last
    const bool mb = s->P.has_en || s->P.n_een > 0;
    const void *k_el = mb ? (d_O ? s->var.b_el_dm : s->var.b_el_m) : (d_O ? s->var.b_el_d : s->var.b_el);
    const void *k_tab = mb ? (d_O ? s->var.b_tab_dm : s->var.b_tab_m) : (d_O ? s->var.b_tab_d : s->var.b_tab);
    auto smem_for = [&](int warps) { return s->P.smem_const_bytes + warps * s->var.bf_ws_doubles * (int)sizeof(double); };
    {
      std::lock_guard<std::mutex> lock(s->scratch_mu);
      if (!s->bf_ready) {
        int dev_smem = 0;
        cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, s->device);
        int we = kWarpsBfTab;  // the explicit kernel: as many warps per block as shared memory holds
        while (we > 1 && smem_for(we) > dev_smem) --we;
        if (smem_for(we) > dev_smem) return QMC_EUNSUPPORTED;
        s->warps_bf = we;
        const int smem = smem_for(we);
        for (const void *k : {s->var.b_el, s->var.b_el_d, s->var.b_el_m, s->var.b_el_dm})
          CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        int per_sm = 0;
        CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, s->var.b_el, we * 32, smem));
        if (per_sm < 1) return QMC_EUNSUPPORTED;
        s->blocks_bf = per_sm * s->n_sm;
        // the table route, for expansions of more than kBfTablesMinDets determinants (measured, CO shape, ms per 32768
        // walkers, tables / explicit: 1 determinant 1.13 / 0.92, 4: 1.43 / 1.11, 20: 1.96 / 2.61, 100: 3.2 / 10.1
        // finds the same for few determinants): as many warps per block (up to kWarpsBfTab) as shared memory holds
        if (s->n_bfdets > kBfTablesMinDets) {
          int wt = kWarpsBfTab;
          while (wt > 1 && s->P.smem_const_bytes + wt * s->var.bf_tab_ws_doubles * (int)sizeof(double) > dev_smem) --wt;
          const int smem_t = s->P.smem_const_bytes + wt * s->var.bf_tab_ws_doubles * (int)sizeof(double);
          if (smem_t <= dev_smem) {
            for (const void *k : {s->var.b_tab, s->var.b_tab_d, s->var.b_tab_m, s->var.b_tab_dm})
              CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_t));
            CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, s->var.b_tab, wt * 32, smem_t));
            if (per_sm >= 1) {
              s->warps_bf_tab = wt;
              s->blocks_bf_tab = per_sm * s->n_sm;
            }
          }
        }
        s->bf_ready = true;
      }
    }
    const int we = s->warps_bf, smem = smem_for(we);
    void *bargs[2] = {(void *)&s->P, (void *)&io};
    if (s->warps_bf_tab > 0 && !explicit_only) {
      // tables first (F.6-F.9), then the explicit kernel over the walkers it listed
      const int wt = s->warps_bf_tab;
      const int grid_t = (int)std::min<int64_t>((M + wt - 1) / wt, s->blocks_bf_tab);
      const size_t e_bytes = (size_t)grid_t * wt * (size_t)s->var.bf_e_doubles * sizeof(double);
      const size_t need = e_bytes + (size_t)(M + 2) * sizeof(int);
      unsigned char *base = nullptr;
      {
        std::lock_guard<std::mutex> lock(s->scratch_mu);
        qmc_system::Scratch &sc = s->scratch[st];
        if (sc.bf_bytes < need) {
          if (sc.bf) s->retired.push_back(sc.bf);
          sc.bf = nullptr;
          sc.bf_bytes = 0;
          CK(cudaMalloc(&sc.bf, need));
          sc.bf_bytes = need;
        }
        base = static_cast<unsigned char *>(sc.bf);
      }
      int *li = reinterpret_cast<int *>(base + e_bytes);
      CK(cudaMemsetAsync(li, 0, sizeof(int), st));
      io.fb_count = li;
      io.fb_list = li + 1;
      const BfDet *dets = static_cast<const BfDet *>(s->d_bfdets);
      double *esc = reinterpret_cast<double *>(base);
      void *targs[5] = {(void *)&s->P, (void *)&io, (void *)&dets, (void *)&s->bf_cls, (void *)&esc};
      const int smem_t = s->P.smem_const_bytes + wt * s->var.bf_tab_ws_doubles * (int)sizeof(double);
      CK(cudaLaunchKernel(k_tab, dim3(grid_t), dim3(wt * 32), targs, smem_t, st));
      ++g_launches;
      CK(cudaLaunchKernel(k_el, dim3(s->blocks_bf), dim3(we * 32), bargs, smem, st));
      ++g_launches;
      return QMC_OK;
    }
    const int grid = (int)std::min<int64_t>((M + we - 1) / we, s->blocks_bf);
    CK(cudaLaunchKernel(k_el, dim3(grid), dim3(we * 32), bargs, smem, st));
    ++g_launches;
    return QMC_OK;
  }
  const int64_t groups = (M + s->P.G - 1) / s->P.G;
  const int wpb = el ? kWarpsEl : s->warps_psi, smem = el ? s->smem_el : s->smem_psi;
  const int64_t need = (groups + wpb - 1) / wpb;
  const int grid = (int)std::min<int64_t>(need, d_O ? s->blocks_deriv : (el ? s->blocks_el : s->blocks_psi));
  double *fb = nullptr;
  const bool fallback = explicit_only || (el && s->P.n_det_all > 1);  // a single determinant has no reference to be ill-conditioned against
  const int64_t expl_warps = (int64_t)s->blocks_expl * kWarpsEl;
  if (fallback) {
    // stream-ordered scratch of the explicit fallback: partial sums [groups + warps][G][2] doubles, then
    // ints: [0] = counter, [1 ..] = listed group indices, then the per-group slice counters
    const size_t n_part = (size_t)(groups + expl_warps) * (size_t)s->P.G * 2;
    const size_t need_bytes = n_part * sizeof(double) + (size_t)(2 * groups + 2) * sizeof(int);
    {
      std::lock_guard<std::mutex> lock(s->scratch_mu);
      qmc_system::Scratch &sc = s->scratch[st];
      if (sc.bytes < need_bytes) {  // grow: the old buffer is kept until qmc_destroy (earlier work on this stream
        if (sc.p) s->retired.push_back(sc.p);  // and graphs captured from earlier calls may still use it)
        sc.p = nullptr;
        sc.bytes = 0;
        CK(cudaMalloc(&sc.p, need_bytes));
        sc.bytes = need_bytes;
      }
      fb = static_cast<double *>(sc.p);
    }
    int *fbi = reinterpret_cast<int *>(fb + n_part);
    CK(cudaMemsetAsync(fbi, 0, sizeof(int), st));
    io.fb_part = fb;
    io.fb_count = fbi;
    io.fb_list = fbi + 1;
    io.fb_done = fbi + 1 + groups;
  }
  void *args[2] = {(void *)&s->P, (void *)&io};
  const bool timed = s->time_kernels && el && !explicit_only;
  if (timed) CK(cudaEventRecord(s->tev[0], st));
  if (explicit_only) {  // every group goes on the list; the table-path kernel is not launched
    if (groups > (int64_t)INT32_MAX) return QMC_EINVAL;
    list_all_groups_kernel<<<(int)std::min<int64_t>((groups + 255) / 256, 1024), 256, 0, st>>>(io.fb_count, io.fb_list, io.fb_done,
                                                                                              (int)groups);
    CK(cudaGetLastError());
  } else {
    CK(cudaLaunchKernel(d_O ? s->var.k_el_deriv : (el ? s->var.k_el : s->var.k_psi), dim3(grid), dim3(wpb * 32), args, smem, st));
  }
  ++g_launches;
  if (timed) CK(cudaEventRecord(s->tev[1], st));
  if (fallback) {
    CK(cudaLaunchKernel(s->var.k_expl, dim3(s->blocks_expl), dim3(kWarpsEl * 32), args, s->smem_el, st));
    ++g_launches;
  }
  if (timed) {
    CK(cudaEventRecord(s->tev[2], st));
    s->tev_fallback = fallback;
  }
  return QMC_OK;
}

int qmc_set_kernel_timing(qmc_system_t *s, int enabled) {
  if (!s) return QMC_EINVAL;
  CK(cudaSetDevice(s->device));
  if (enabled)
    for (cudaEvent_t &e : s->tev)
      if (!e) CK(cudaEventCreate(&e));
  s->time_kernels = enabled != 0;
  return QMC_OK;
}

int qmc_kernel_times(qmc_system_t *s, double *h_main_ms, double *h_fallback_ms) {
  if (!s || !s->tev[2]) return QMC_EINVAL;
  CK(cudaSetDevice(s->device));
  CK(cudaEventSynchronize(s->tev[2]));
  float a = 0.f, b = 0.f;
  CK(cudaEventElapsedTime(&a, s->tev[0], s->tev[1]));
  CK(cudaEventElapsedTime(&b, s->tev[1], s->tev[2]));
  if (h_main_ms) *h_main_ms = a;
  if (h_fallback_ms) *h_fallback_ms = s->tev_fallback ? b : 0.0;
  return QMC_OK;
}

int qmc_local_energy(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign, double *d_eloc,
                     void *cuda_stream) {
  return launch_eval(s, d_r, M, d_logpsi, d_sign, d_eloc, cuda_stream, true);
}

int qmc_local_energy_explicit(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign,
                              double *d_eloc, void *cuda_stream) {
  return launch_eval(s, d_r, M, d_logpsi, d_sign, d_eloc, cuda_stream, true, nullptr, true);
}

int qmc_local_energy_host(qmc_system_t *s, const double *h_r, int64_t M, double *h_logpsi, double *h_sign,
                          double *h_eloc, int32_t n_chunks) {
  if (!s || !h_r || M <= 0 || n_chunks < 1) return QMC_EINVAL;
  CK(cudaSetDevice(s->device));
  const int ne = s->P.n_e;
  int64_t Mc = (M + n_chunks - 1) / n_chunks;
  Mc = (Mc + 31) / 32 * 32;  // whole warps' worth of groups per chunk
  if (Mc > s->hbuf_walkers) {  // [3 n_e + 3][Mc] doubles per buffer: coordinates, then log|Psi|, sign, E_L
    for (int i = 0; i < 2; ++i) {
      if (!s->hst[i]) CK(cudaStreamCreateWithFlags(&s->hst[i], cudaStreamNonBlocking));
      CK(cudaStreamSynchronize(s->hst[i]));
      cudaFree(s->hbuf[i]);
      s->hbuf[i] = nullptr;
      CK(cudaMalloc(&s->hbuf[i], (size_t)(3 * ne + 3) * (size_t)Mc * sizeof(double)));
    }
    s->hbuf_walkers = Mc;
  }
  int rc = QMC_OK;
  int c = 0;
  for (int64_t a = 0; a < M && rc == QMC_OK; a += Mc, ++c) {
    const int64_t m = std::min<int64_t>(Mc, M - a);
    cudaStream_t st = s->hst[c & 1];
    double *d_r = s->hbuf[c & 1], *d_out = d_r + (size_t)3 * ne * (size_t)m;
    // rows of the SoA array are M doubles apart on the host and m doubles apart in the chunk buffer
    CK(cudaMemcpy2DAsync(d_r, (size_t)m * sizeof(double), h_r + a, (size_t)M * sizeof(double), (size_t)m * sizeof(double),
                         (size_t)3 * ne, cudaMemcpyHostToDevice, st));
    rc = launch_eval(s, d_r, m, h_logpsi ? d_out : nullptr, h_sign ? d_out + m : nullptr, h_eloc ? d_out + 2 * m : nullptr,
                     st, true);
    if (rc != QMC_OK) break;
    if (h_logpsi) CK(cudaMemcpyAsync(h_logpsi + a, d_out, (size_t)m * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (h_sign) CK(cudaMemcpyAsync(h_sign + a, d_out + m, (size_t)m * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (h_eloc) CK(cudaMemcpyAsync(h_eloc + a, d_out + 2 * m, (size_t)m * sizeof(double), cudaMemcpyDeviceToHost, st));
  }
  for (int i = 0; i < 2; ++i)
    if (s->hst[i]) {
      cudaError_t e = cudaStreamSynchronize(s->hst[i]);
      if (e != cudaSuccess && rc == QMC_OK) rc = cuda_fail(e, "qmc_local_energy_host");
    }
  return rc;
}

int qmc_vmc_step_host(qmc_system_t *s, double *h_r, int64_t M, double step, int32_t n_sweeps, uint64_t seed,
                      uint64_t sweep_offset, int64_t walker_offset, double *h_eloc, double *h_mean, double *h_stderr,
                      int32_t n_chunks) {
  if (!s || !h_r || M <= 0 || n_chunks < 1 || !(step > 0.0) || n_sweeps < 0 || walker_offset < 0) return QMC_EINVAL;
  CK(cudaSetDevice(s->device));
  const int ne = s->P.n_e;
  int64_t Mc = (M + n_chunks - 1) / n_chunks;
  Mc = (Mc + 31) / 32 * 32;
  if (Mc > s->hbuf_walkers) {
    for (int i = 0; i < 2; ++i) {
      if (!s->hst[i]) CK(cudaStreamCreateWithFlags(&s->hst[i], cudaStreamNonBlocking));
      CK(cudaStreamSynchronize(s->hst[i]));
      cudaFree(s->hbuf[i]);
      s->hbuf[i] = nullptr;
      CK(cudaMalloc(&s->hbuf[i], (size_t)(3 * ne + 3) * (size_t)Mc * sizeof(double)));
    }
    s->hbuf_walkers = Mc;
  }
  if (M > s->helo_walkers) {
    CK(cudaDeviceSynchronize());
    cudaFree(s->helo);
    s->helo = nullptr;
    CK(cudaMalloc(&s->helo, (size_t)M * sizeof(double)));
    s->helo_walkers = M;
  }
  int rc = QMC_OK;
  int c = 0;
  for (int64_t a = 0; a < M && rc == QMC_OK; a += Mc, ++c) {
    const int64_t m = std::min<int64_t>(Mc, M - a);
    cudaStream_t st = s->hst[c & 1];
    double *d_r = s->hbuf[c & 1];
    CK(cudaMemcpy2DAsync(d_r, (size_t)m * sizeof(double), h_r + a, (size_t)M * sizeof(double), (size_t)m * sizeof(double),
                         (size_t)3 * ne, cudaMemcpyHostToDevice, st));
    rc = qmc_metropolis(s, d_r, m, step, n_sweeps, seed, sweep_offset, walker_offset + a, nullptr, nullptr, nullptr, nullptr,
                        nullptr, st);
    if (rc != QMC_OK) break;
    rc = launch_eval(s, d_r, m, nullptr, nullptr, s->helo + a, st, true);
    if (rc != QMC_OK) break;
    CK(cudaMemcpy2DAsync(h_r + a, (size_t)M * sizeof(double), d_r, (size_t)m * sizeof(double), (size_t)m * sizeof(double),
                         (size_t)3 * ne, cudaMemcpyDeviceToHost, st));
    if (h_eloc) CK(cudaMemcpyAsync(h_eloc + a, s->helo + a, (size_t)m * sizeof(double), cudaMemcpyDeviceToHost, st));
  }
  for (int i = 0; i < 2; ++i)
    if (s->hst[i]) {
      cudaError_t e = cudaStreamSynchronize(s->hst[i]);
      if (e != cudaSuccess && rc == QMC_OK) rc = cuda_fail(e, "qmc_vmc_step_host");
    }
  if (rc == QMC_OK && (h_mean || h_stderr)) rc = qmc_batch_stats(s->helo, M, h_mean, h_stderr, s->hst[0]);
  return rc;
}

int qmc_log_psi(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign, void *cuda_stream) {
  return launch_eval(s, d_r, M, d_logpsi, d_sign, nullptr, cuda_stream, false);
}

int qmc_metropolis(qmc_system_t *s, double *d_r, int64_t M, double step, int32_t n_sweeps, uint64_t seed,
                   uint64_t sweep_offset, int64_t walker_offset, double *d_logpsi, double *d_sign, uint8_t *d_accept,
                   double *d_eloc_acc, int64_t *h_n_accepted, void *cuda_stream) {
  if (!s || !d_r || M <= 0 || !(step > 0.0) || n_sweeps < 0 || walker_offset < 0) return QMC_EINVAL;
  if (sweep_offset + (uint64_t)n_sweeps >= (1ull << 32)) return QMC_EINVAL;
  CK(cudaSetDevice(s->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  WalkerIO io{};
  io.r_in = d_r;
  io.r_out = d_r;
  io.logpsi = d_logpsi;
  io.sign = d_sign;
  io.M = M;
  MetroParams mp{};
  mp.step = step;
  mp.n_sweeps = n_sweeps;
  mp.key0 = (uint32_t)(seed & 0xFFFFFFFFu);
  mp.key1 = (uint32_t)(seed >> 32);
  mp.sweep0 = (uint32_t)sweep_offset;
  mp.walker_offset = walker_offset;
  mp.accept = d_accept;
  mp.resume = 0;
  unsigned long long *d_counter = nullptr;
  if (h_n_accepted) {  // the accept counter belongs to the calling stream
    std::lock_guard<std::mutex> lock(s->scratch_mu);
    qmc_system::Scratch &sc = s->scratch[st];
    if (!sc.counter) CK(cudaMalloc(&sc.counter, sizeof(unsigned long long)));
    d_counter = sc.counter;
  }
  mp.n_accepted = d_counter;
  if (h_n_accepted) CK(cudaMemsetAsync(d_counter, 0, sizeof(unsigned long long), st));
  const int64_t groups = (M + s->P.G - 1) / s->P.G;
  const int64_t need = (groups + s->warps_metro - 1) / s->warps_metro;
  const int grid = (int)std::min<int64_t>(need, s->blocks_metro);
  void *args[3] = {(void *)&s->P, (void *)&io, (void *)&mp};
  if (!d_eloc_acc) {
    // one persistent launch for all sweeps: coordinates and log|Psi| stay in registers
    CK(cudaLaunchKernel(s->var.k_metro, dim3(grid), dim3(s->warps_metro * 32), args, s->smem_metro, st));
    ++g_launches;
  } else {
    // E_L after every sweep (BASELINE config 5): one-sweep launches of the sampler alternate with the
    // local-energy call (fast kernel + explicit fallback), whose result is added to d_eloc_acc.  The
    // sampler resumes from the log|Psi| / sign the previous launch stored, so no evaluation is repeated.
    double *scratch = nullptr;  // [M] E_L of one sweep, then [M] log|Psi|, [M] sign if the caller gave none
    const size_t n_scr = (size_t)M * (1 + (d_logpsi ? 0 : 1) + (d_sign ? 0 : 1));
    CK(cudaMallocAsync(&scratch, n_scr * sizeof(double), st));
    // every failure below releases the scratch before returning
#define CKS(call)                                          \
  do {                                                     \
    cudaError_t e__ = (call);                              \
    if (e__ != cudaSuccess) {                              \
      cudaFreeAsync(scratch, st);                          \
      return cuda_fail(e__, #call);                        \
    }                                                      \
  } while (0)
    double *nxt = scratch + M;
    if (!d_logpsi) { io.logpsi = nxt; nxt += M; }
    if (!d_sign) io.sign = nxt;
    CKS(cudaMemsetAsync(d_eloc_acc, 0, (size_t)M * sizeof(double), st));
    mp.n_sweeps = 1;
    if (n_sweeps == 0) {  // nothing to accumulate; still report log|Psi| of the starting positions
      mp.n_sweeps = 0;
      CKS(cudaLaunchKernel(s->var.k_metro, dim3(grid), dim3(s->warps_metro * 32), args, s->smem_metro, st));
      ++g_launches;
    }
    for (int32_t sw = 0; sw < n_sweeps; ++sw) {
      mp.sweep0 = (uint32_t)(sweep_offset + (uint64_t)sw);
      mp.accept = d_accept ? d_accept + (size_t)sw * (size_t)M : nullptr;
      mp.resume = sw > 0 ? 1 : 0;
      CKS(cudaLaunchKernel(s->var.k_metro, dim3(grid), dim3(s->warps_metro * 32), args, s->smem_metro, st));
      ++g_launches;
      int rc = launch_eval(s, d_r, M, nullptr, nullptr, scratch, st, true);
      if (rc != QMC_OK) {
        cudaFreeAsync(scratch, st);
        return rc;
      }
      accumulate_kernel<<<(unsigned)std::min<int64_t>((M + 255) / 256, 4 * s->n_sm), 256, 0, st>>>(d_eloc_acc, scratch, M);
      CKS(cudaGetLastError());
      ++g_launches;
    }
#undef CKS
    CK(cudaFreeAsync(scratch, st));
  }
  if (h_n_accepted) {
    unsigned long long v = 0;
    CK(cudaMemcpyAsync(&v, d_counter, sizeof(v), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    *h_n_accepted = (int64_t)v;
  }
  return QMC_OK;
}

int qmc_n_param(const qmc_system_t *s) {
  return s ? kJastrowParams + 7 * s->P.n_een + s->P.n_det_all + (s->P.bf_w != 0.0 ? 1 : 0) : QMC_EINVAL;  // backflow: + its weight
}

int qmc_log_derivatives(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign, double *d_eloc,
                        double *d_O, void *cuda_stream) {
  if (!d_O) return QMC_EINVAL;
  return launch_eval(s, d_r, M, d_logpsi, d_sign, d_eloc, cuda_stream, true, d_O);
}

int qmc_energy_gradient(const double *d_eloc, const double *d_O, int64_t M, int32_t n_param, double *h_Ev, double *h_grad,
                        void *cuda_stream) {
  if (!d_eloc || !d_O || M <= 0 || n_param < 1 || !h_grad) return QMC_EINVAL;
  int dev = 0;
  if (int rc = device_of(d_eloc, &dev)) return rc;
  CK(cudaSetDevice(dev));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nblk = (int)std::min<int64_t>(1184, (M + 63) / 64);  // >= 64 rows per block
  ReduceScratch *r = nullptr;
  if (int rc = reduce_scratch(dev, st, (size_t)n_param, (size_t)nblk * (size_t)n_param, &r)) return rc;
  const int sblk = (int)std::min<int64_t>(kReduceBlocks, (M + kStatsThreads - 1) / kStatsThreads);
  batch_stats_kernel<<<sblk, kStatsThreads, 0, st>>>(d_eloc, M, r->d_partial, r->d_done, r->d_stats);
  CK(cudaGetLastError());
  gradient_partial_kernel<<<nblk, 128, 0, st>>>(d_eloc, d_O, M, n_param, r->d_stats, r->d_gpart);
  CK(cudaGetLastError());
  gradient_final_kernel<<<n_param, 128, 0, st>>>(r->d_gpart, nblk, n_param, M, r->d_stats, r->d_res);
  CK(cudaGetLastError());
  g_launches += 3;
  CK(cudaStreamSynchronize(st));  // the final kernel wrote {E_v, stderr, grad[...]} into mapped host memory
  if (h_Ev) *h_Ev = r->h_res[0];
  for (int p = 0; p < n_param; ++p) h_grad[p] = r->h_res[2 + p];
  return QMC_OK;
}

// one launch of orbital_derivatives_kernel: (dC, dzeta) or, with d_dR, the AO part of the nuclear log-gradient
static int orbital_launch(qmc_system_t *s, const double *d_r, int64_t M, double *d_dC, double *d_dzeta, double *d_dR,
                          void *cuda_stream) {
  CK(cudaSetDevice(s->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  auto smem_for = [&](int warps) { return s->P.smem_const_bytes + warps * s->var.orb_ws_doubles * (int)sizeof(double); };
  std::lock_guard<std::mutex> lock(s->scratch_mu);  // lazy configuration; the launch below is asynchronous
  if (!s->orb_ready) {
    int dev_smem = 0;
    cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, s->device);
    s->orb_warps = smem_for(kWarpsOrb) <= dev_smem ? kWarpsOrb : kWarpsOrbSmall;
    if (smem_for(s->orb_warps) > dev_smem) return QMC_EUNSUPPORTED;
    const void *k = s->orb_warps == kWarpsOrb ? s->var.k_orb : s->var.k_orb_small;
    CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_for(s->orb_warps)));
    CK(cudaFuncSetAttribute(s->orb_warps == kWarpsOrb ? s->var.k_nuc : s->var.k_nuc_small,
                            cudaFuncAttributeMaxDynamicSharedMemorySize, smem_for(s->orb_warps)));
    CK(cudaFuncSetAttribute(s->orb_warps == kWarpsOrb ? s->var.x_orb : s->var.x_orb_small,
                            cudaFuncAttributeMaxDynamicSharedMemorySize, smem_for(s->orb_warps)));
    CK(cudaFuncSetAttribute(s->orb_warps == kWarpsOrb ? s->var.x_nuc : s->var.x_nuc_small,
                            cudaFuncAttributeMaxDynamicSharedMemorySize, smem_for(s->orb_warps)));
    int per_sm = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, s->orb_warps * 32, smem_for(s->orb_warps)));
    if (per_sm < 1) return QMC_EUNSUPPORTED;
    s->blocks_orb = per_sm * s->n_sm;
    s->orb_ready = true;
  }
  const int warps = s->orb_warps, smem = smem_for(warps);
  const void *kern = d_dR ? (warps == kWarpsOrb ? s->var.k_nuc : s->var.k_nuc_small)
                          : (warps == kWarpsOrb ? s->var.k_orb : s->var.k_orb_small);
  // coefficients of MOs that no determinant uses have a zero derivative and are not touched by the kernel
  if (d_dC && s->P.n_mo < s->P.n_mo_all) CK(cudaMemsetAsync(d_dC, 0, (size_t)M * (size_t)s->P.n_ao * (size_t)s->P.n_mo_all * sizeof(double), st));
  WalkerIO io{};
  io.r_in = d_r;
  io.M = M;
  io.logpsi = d_dC;    // this kernel's outputs travel in the two output slots: dC [M][n_ao][n_mo], dzeta [M][n_ao]
  io.eloc = d_dzeta;
  io.O = d_dR;         // nuclear mode: dR [M][n_atoms][3], decremented by the AO part
  const int64_t groups = (M + s->P.G - 1) / s->P.G;
  const int grid = (int)std::min<int64_t>((groups + warps - 1) / warps, s->blocks_orb);
  {
    // scratch of the pair of launches: {work counter, list counter}; the listed groups' partial Gamma per work item of the
    // explicit kernel (at most one item per warp of its grid when a group is sliced), the group list and slice counters
    qmc_system::Scratch &sc = s->scratch[st];  // (scratch_mu is held)
    if (!sc.work) CK(cudaMalloc(&sc.work, 2 * sizeof(int)));
    io.fb_count = sc.work;
    const size_t ps = (size_t)s->P.G * (size_t)s->P.n_e * (size_t)s->var.NMO + (size_t)s->P.G;
    const size_t n_part = (size_t)s->blocks_orb * (size_t)warps * ps;
    const size_t need = n_part * sizeof(double) + (size_t)(2 * groups) * sizeof(int);
    if (sc.orb_bytes < need) {
      if (sc.orb) s->retired.push_back(sc.orb);
      sc.orb = nullptr;
      sc.orb_bytes = 0;
      CK(cudaMalloc(&sc.orb, need));
      sc.orb_bytes = need;
    }
    io.fb_part = static_cast<double *>(sc.orb);
    io.fb_list = reinterpret_cast<int *>(io.fb_part + n_part);
    io.fb_done = io.fb_list + groups;
  }
  CK(cudaMemsetAsync(io.fb_count, 0, 2 * sizeof(int), st));
  void *args[2] = {(void *)&s->P, (void *)&io};
  CK(cudaLaunchKernel(kern, dim3(grid), dim3(warps * 32), args, smem, st));
  const void *kx = d_dR ? (warps == kWarpsOrb ? s->var.x_nuc : s->var.x_nuc_small)
                        : (warps == kWarpsOrb ? s->var.x_orb : s->var.x_orb_small);
  CK(cudaLaunchKernel(kx, dim3(s->blocks_orb), dim3(warps * 32), args, smem, st));
  g_launches += 2;
  return QMC_OK;
}

int qmc_orbital_derivatives(qmc_system_t *s, const double *d_r, int64_t M, double *d_dC, double *d_dzeta, void *cuda_stream) {
  if (!s || !d_r || M <= 0 || (!d_dC && !d_dzeta)) return QMC_EINVAL;
  return orbital_launch(s, d_r, M, d_dC, d_dzeta, nullptr, cuda_stream);
}

int qmc_nuclear_log_gradient(qmc_system_t *s, const double *d_r, int64_t M, double *d_dR, void *cuda_stream) {
  if (!s || !d_r || M <= 0 || !d_dR) return QMC_EINVAL;
  CK(cudaSetDevice(s->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // Jastrow part (D.2, D.3) initialises dR, one thread per walker; the AO part is subtracted by the second launch
  nuclear_jastrow_gradient_kernel<<<(unsigned)((M + 127) / 128), 128, 0, st>>>(s->P, d_r, M, d_dR);
  CK(cudaGetLastError());
  ++g_launches;
  return orbital_launch(s, d_r, M, nullptr, nullptr, d_dR, cuda_stream);
}

int qmc_local_energy_gradient(qmc_system_t *s, const double *d_r, int64_t M, double *d_logpsi, double *d_sign, double *d_eloc,
                              double *h_Ev, double *h_grad, void *cuda_stream) {
  if (!s || !d_r || M <= 0 || !d_eloc || !h_grad) return QMC_EINVAL;
  CK(cudaSetDevice(s->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (s->P.bf_w != 0.0) {
    // backflow wavefunction: the same estimator from qmc_log_derivatives and qmc_energy_gradient, the rows [M][n_param]
    // in a per-stream scratch of the handle (not fused: the backflow kernels hold one walker per warp and no row buffer)
    const int npb = qmc_n_param(s);
    const size_t need = (size_t)M * (size_t)npb * sizeof(double);
    double *rows = nullptr;
    {
      std::lock_guard<std::mutex> lock(s->scratch_mu);
      qmc_system::Scratch &sc = s->scratch[st];
      if (sc.fuse_bytes < need) {
        if (sc.fuse) s->retired.push_back(sc.fuse);
        sc.fuse = nullptr;
        sc.fuse_bytes = 0;
        CK(cudaMalloc(&sc.fuse, need));
        sc.fuse_bytes = need;
      }
      rows = static_cast<double *>(sc.fuse);
    }
    if (int rc = launch_eval(s, d_r, M, d_logpsi, d_sign, d_eloc, cuda_stream, true, rows)) return rc;
    return qmc_energy_gradient(d_eloc, rows, M, npb, h_Ev, h_grad, cuda_stream);
  }
  const int np = kJastrowParams + 7 * s->P.n_een + s->P.n_det_all, G = s->P.G;
  const int fuse_stride = ((G + 2) * np + G + 1) & ~1;  // G rows, two accumulator rows, 1 / (Sigma / D_0) per walker
  const void *kern = s->P.n_een > 0 ? s->var.e_el_fuse : s->var.k_el_fuse;
  {
    std::lock_guard<std::mutex> lock(s->scratch_mu);  // lazy configuration
    if (!s->fuse_ready) {
      int dev_smem = 0;
      cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, s->device);
      s->smem_fuse = s->smem_el + kWarpsEl * fuse_stride * (int)sizeof(double);
      if (s->smem_fuse > dev_smem) return QMC_EUNSUPPORTED;  // too many parameters for the fused rows: use qmc_log_derivatives
      CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, s->smem_fuse));
      int per_sm = 0;
      CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kWarpsEl * 32, s->smem_fuse));
      if (per_sm < 1) return QMC_EUNSUPPORTED;
      s->blocks_fuse = per_sm * s->n_sm;
      s->fuse_ready = true;
    }
  }
  const int64_t groups = (M + G - 1) / G;
  const int grid = (int)std::min<int64_t>((groups + kWarpsEl - 1) / kWarpsEl, s->blocks_fuse);
  const int n_warps = grid * kWarpsEl;
  const bool fallback = s->P.n_det_all > 1;
  const int cap = (int)std::min<int64_t>(groups, 8192);
  // scratch of the explicit fallback (as qmc_local_energy) and of the fused reduction, both per stream
  const int64_t expl_warps = (int64_t)s->blocks_expl * kWarpsEl;
  const size_t n_part = (size_t)(groups + expl_warps) * (size_t)G * 2;
  const size_t need_fb = n_part * sizeof(double) + (size_t)(2 * groups + 2) * sizeof(int);
  const size_t n_fpart = (size_t)n_warps * (size_t)(2 * np + 2), n_fbO = (size_t)cap * (size_t)G * (size_t)np;
  const size_t need_fuse = (n_fpart + n_fbO) * sizeof(double) + (size_t)(cap + 2) * sizeof(int);
  double *fb = nullptr, *fz = nullptr;
  {
    std::lock_guard<std::mutex> lock(s->scratch_mu);
    qmc_system::Scratch &sc = s->scratch[st];
    if (sc.bytes < need_fb) {
      if (sc.p) s->retired.push_back(sc.p);
      sc.p = nullptr;
      sc.bytes = 0;
      CK(cudaMalloc(&sc.p, need_fb));
      sc.bytes = need_fb;
    }
    if (sc.fuse_bytes < need_fuse) {
      if (sc.fuse) s->retired.push_back(sc.fuse);
      sc.fuse = nullptr;
      sc.fuse_bytes = 0;
      CK(cudaMalloc(&sc.fuse, need_fuse));
      sc.fuse_bytes = need_fuse;
    }
    fb = static_cast<double *>(sc.p);
    fz = static_cast<double *>(sc.fuse);
  }
  int dev = s->device;
  ReduceScratch *rs = nullptr;
  if (int rc = reduce_scratch(dev, st, (size_t)np, 0, &rs)) return rc;
  int *fbi = reinterpret_cast<int *>(fb + n_part);
  int *fzi = reinterpret_cast<int *>(fz + n_fpart + n_fbO);  // [0] = overflow flag, [1 ..] = order
  CK(cudaMemsetAsync(fbi, 0, sizeof(int), st));
  CK(cudaMemsetAsync(fzi, 0, sizeof(int), st));
  WalkerIO io{};
  io.r_in = d_r;
  io.logpsi = d_logpsi;
  io.sign = d_sign;
  io.eloc = d_eloc;
  io.M = M;
  io.fuse_part = fz;
  io.fb_O = fz + n_fpart;
  io.fb_cap = cap;
  io.fb_over = fzi;
  io.fuse_stride = fuse_stride;
  if (fallback) {
    io.fb_part = fb;
    io.fb_count = fbi;
    io.fb_list = fbi + 1;
    io.fb_done = fbi + 1 + groups;
  }
  void *args[2] = {(void *)&s->P, (void *)&io};
  CK(cudaLaunchKernel(kern, dim3(grid), dim3(kWarpsEl * 32), args, s->smem_fuse, st));
  ++g_launches;
  if (fallback) {
    CK(cudaLaunchKernel(s->var.k_expl, dim3(s->blocks_expl), dim3(kWarpsEl * 32), args, s->smem_el, st));
    order_flagged_kernel<<<1, 1024, 0, st>>>(io.fb_count, io.fb_list, cap, fzi + 1);
    CK(cudaGetLastError());
    g_launches += 2;
  }
  fused_gradient_final_kernel<<<np, 128, 0, st>>>(fz, n_warps, np, fallback ? io.fb_count : nullptr, io.fb_list, fzi + 1, io.fb_O, cap,
                                                d_eloc, G, M, kJastrowParams + 7 * s->P.n_een, s->P.det_orig, fzi, rs->d_res);
  CK(cudaGetLastError());
  ++g_launches;
  CK(cudaStreamSynchronize(st));  // the final kernel wrote {E_v, overflow flag, grad} into mapped host memory
  if (rs->h_res[1] != 0.0) {
    // more groups took the explicit route than the parking area holds (pathological batch): the unfused path
    double *d_O = nullptr;
    CK(cudaMalloc(&d_O, (size_t)M * (size_t)np * sizeof(double)));
    int rc = launch_eval(s, d_r, M, d_logpsi, d_sign, d_eloc, cuda_stream, true, d_O);
    if (rc == QMC_OK) rc = qmc_energy_gradient(d_eloc, d_O, M, np, h_Ev, h_grad, cuda_stream);
    cudaFree(d_O);
    return rc;
  }
  if (h_Ev) *h_Ev = rs->h_res[0];
  for (int p = 0; p < np; ++p) h_grad[p] = rs->h_res[2 + p];
  return QMC_OK;
}

int qmc_nuclear_energy_gradient(qmc_system_t *s, const double *d_r, int64_t M, double *d_dE, void *cuda_stream) {
  if (!s || !d_r || M <= 0 || !d_dE) return QMC_EINVAL;
  if (s->P.has_en || s->P.n_een > 0 || s->P.bf_w != 0.0) return QMC_EUNSUPPORTED;  // D.2 / D.3 / backflow inside E_L: not derived
  CK(cudaSetDevice(s->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  auto smem_for = [&](int warps) { return s->P.smem_const_bytes + warps * s->var.frc_ws_doubles * (int)sizeof(double); };
  {
    std::lock_guard<std::mutex> lock(s->scratch_mu);  // lazy configuration
    if (!s->frc_ready) {
      int dev_smem = 0;
      cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, s->device);
      s->frc_warps = smem_for(8) <= dev_smem ? 8 : 4;
      if (smem_for(s->frc_warps) > dev_smem) return QMC_EUNSUPPORTED;
      const void *k = s->frc_warps == 8 ? s->var.k_frc : s->var.k_frc_small;
      CK(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_for(s->frc_warps)));
      int per_sm = 0;
      CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, s->frc_warps * 32, smem_for(s->frc_warps)));
      if (per_sm < 1) return QMC_EUNSUPPORTED;
      s->blocks_frc = per_sm * s->n_sm;
      s->frc_ready = true;
    }
  }
  // d V / d R initialises dE, one thread per walker; the wavefunction part is added by the second launch
  nuclear_potential_gradient_kernel<<<(unsigned)((M + 127) / 128), 128, 0, st>>>(s->P, d_r, M, d_dE);
  CK(cudaGetLastError());
  ++g_launches;
  WalkerIO io{};
  io.r_in = d_r;
  io.M = M;
  io.O = d_dE;
  {
    std::lock_guard<std::mutex> lock(s->scratch_mu);
    qmc_system::Scratch &sc = s->scratch[st];
    if (!sc.work) CK(cudaMalloc(&sc.work, 2 * sizeof(int)));
    io.fb_count = sc.work;
  }
  CK(cudaMemsetAsync(io.fb_count, 0, sizeof(int), st));
  const int warps = s->frc_warps;
  const int64_t groups = (M + s->P.G - 1) / s->P.G;
  const int grid = (int)std::min<int64_t>((groups + warps - 1) / warps, s->blocks_frc);
  void *args[2] = {(void *)&s->P, (void *)&io};
  CK(cudaLaunchKernel(warps == 8 ? s->var.k_frc : s->var.k_frc_small, dim3(grid), dim3(warps * 32), args, smem_for(warps), st));
  ++g_launches;
  return QMC_OK;
}

int qmc_force(const double *d_eloc, const double *d_dE, const double *d_dlnpsi, int64_t M, int32_t n_atoms, double *h_F,
              double *h_terms, void *cuda_stream) {
  if (!d_eloc || !d_dE || !d_dlnpsi || M <= 0 || n_atoms < 1 || !h_F) return QMC_EINVAL;
  int dev = 0;
  if (int rc = device_of(d_eloc, &dev)) return rc;
  CK(cudaSetDevice(dev));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nc = 3 * n_atoms;
  const int nblk = (int)std::min<int64_t>(1184, (M + 63) / 64);
  ReduceScratch *r = nullptr;
  if (int rc = reduce_scratch(dev, st, (size_t)2 * nc, (size_t)nblk * 2 * (size_t)nc, &r)) return rc;
  const int sblk = (int)std::min<int64_t>(kReduceBlocks, (M + kStatsThreads - 1) / kStatsThreads);
  batch_stats_kernel<<<sblk, kStatsThreads, 0, st>>>(d_eloc, M, r->d_partial, r->d_done, r->d_stats);
  CK(cudaGetLastError());
  force_partial_kernel<<<nblk, 128, 0, st>>>(d_eloc, d_dE, d_dlnpsi, M, nc, r->d_stats, r->d_gpart);
  CK(cudaGetLastError());
  force_final_kernel<<<2 * nc, 128, 0, st>>>(r->d_gpart, nblk, nc, M, r->d_stats, r->d_res);
  CK(cudaGetLastError());
  g_launches += 3;
  CK(cudaStreamSynchronize(st));
  for (int j = 0; j < nc; ++j) {
    const double t1 = r->h_res[2 + j], t2 = r->h_res[2 + nc + j];
    h_F[j] = t1 + t2;
    if (h_terms) { h_terms[j] = t1; h_terms[nc + j] = t2; }
  }
  return QMC_OK;
}

int qmc_batch_stats(const double *d_x, int64_t M, double *h_mean, double *h_stderr, void *cuda_stream) {
  if (!d_x || M <= 0) return QMC_EINVAL;
  int dev = 0;
  if (int rc = device_of(d_x, &dev)) return rc;
  CK(cudaSetDevice(dev));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  ReduceScratch *r = nullptr;
  if (int rc = reduce_scratch(dev, st, 0, 0, &r)) return rc;
  const int nblk = (int)std::min<int64_t>(kReduceBlocks, (M + kStatsThreads - 1) / kStatsThreads);
  batch_stats_kernel<<<nblk, kStatsThreads, 0, st>>>(d_x, M, r->d_partial, r->d_done, r->d_res);
  CK(cudaGetLastError());
  ++g_launches;
  CK(cudaStreamSynchronize(st));  // the last block wrote {mean, stderr} into mapped host memory
  if (h_mean) *h_mean = r->h_res[0];
  if (h_stderr) *h_stderr = r->h_res[1];
  return QMC_OK;
}

int qmc_static_scratch_init(int device) {
  if (device < 0 || device >= kStaticMaxDevices) return QMC_EINVAL;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (g_static_ptr[device]) return QMC_OK;
  CK(cudaSetDevice(device));
  unsigned char *ptr = nullptr;
  CK(cudaGetSymbolAddress((void **)&ptr, g_static_scratch));  // with `device` current: this device's copy of the array
  if (!ptr) return QMC_ECUDA;
  g_static_ptr[device] = ptr;
  return QMC_OK;
}

int qmc_batch_stats_static(const double *d_x, int64_t M, double *d_out, void *cuda_stream) {
  if (!d_x || !d_out || M <= 0) return QMC_EINVAL;
  if (M > kStaticMaxM) return QMC_ETOOLARGE;  // beyond the fixed scratch's stated limit
  int dev = 0;
  if (int rc = device_of(d_x, &dev)) return rc;
  if (dev < 0 || dev >= kStaticMaxDevices) return QMC_EINVAL;
  if (!g_static_ptr[dev])
    if (int rc = qmc_static_scratch_init(dev)) return rc;
  CK(cudaSetDevice(dev));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  unsigned char *base = g_static_ptr[dev];
  double *partial = reinterpret_cast<double *>(base);
  unsigned int *done = reinterpret_cast<unsigned int *>(base + kStaticPartialBytes);
  // the array keeps the last call's contents: the counter must start at zero (the partials are overwritten before read)
  CK(cudaMemsetAsync(done, 0, sizeof(unsigned int), st));
  const int nblk = (int)std::min<int64_t>(kStaticBlocks, (M + kStatsThreads - 1) / kStatsThreads);
  batch_stats_kernel<<<nblk, kStatsThreads, 0, st>>>(d_x, M, partial, done, d_out);
  CK(cudaGetLastError());
  ++g_launches;
  return QMC_OK;
}

int qmc_fp64_peak(int device, int kind, int reps, double *h_tflops) {
  if (!h_tflops || kind < 0 || kind > 5 || reps < 1) return QMC_EINVAL;
  CK(cudaSetDevice(device));
  int n_sm = 0;
  CK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device));
  double *d_out = nullptr;
  CK(cudaMalloc(&d_out, sizeof(double)));
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0));
  CK(cudaEventCreate(&e1));
  const int iters = 4096, threads = (kind == 5) ? 128 : 256;  // kind 5: one warp per SM sub-partition
  const int blocks = (kind == 5) ? n_sm : n_sm * 8;
  double best = 0.0;
  for (int r = 0; r < reps + 1; ++r) {
    CK(cudaEventRecord(e0, 0));
    if (kind == 0) fp64_peak_kernel<0><<<blocks, threads>>>(d_out, iters, 1.0);
    if (kind == 1) fp64_peak_kernel<1><<<blocks, threads>>>(d_out, iters, 1.0);
    if (kind == 2) fp64_peak_kernel<2><<<blocks, threads>>>(d_out, iters, 1.0);
    if (kind == 3) fp64_probe_kernel<3><<<blocks, threads>>>(d_out, iters, 1.0);
    if (kind == 4) fp64_probe_kernel<4><<<blocks, threads>>>(d_out, iters, 1.0);
    if (kind == 5) fp64_probe_kernel<5><<<blocks, threads>>>(d_out, iters, 1.0);
    ++g_launches;
    CK(cudaEventRecord(e1, 0));
    CK(cudaEventSynchronize(e1));
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    double flops_thread = 0;
    if (kind == 0 || kind == 2 || kind >= 3) flops_thread += (double)iters * 32 * 2;
    if (kind == 1 || kind == 2) flops_thread += (double)iters * 4 * 512 / 32;
    const double tf = flops_thread * blocks * threads / (ms * 1e-3) / 1e12;
    if (r > 0 && tf > best) best = tf;  // first launch is warm-up
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d_out);
  *h_tflops = best;
  return QMC_OK;
}

double qmc_model_flops(const qmc_system_t *s, int which) {
  if (!s) return 0.0;
  return which == 0 ? s->flops_el : s->flops_step;
}

}  // extern "C"
