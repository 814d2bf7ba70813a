// qmc_variant.cuh -- one compiled (NS, NMO) instantiation of the template kernels as a table of entry points.
// Each instantiation lives in its own translation unit (qmc_variant_*.cu, which define QMC_VARIANT_TU and
// QMC_VARIANT_ARGS), so that the build compiles them in parallel; qmc_api.cu only collects the tables.
#pragma once
#include "qmc_kernels.cuh"

namespace qmc {

struct Variant {
  int NS, NMO, LP, ws_doubles;
  int wpb_psi_max;       // launch bound of the values-only kernels, in warps
  int psi_ws_doubles;    // the values-only kernels' compact scratch
  int metro_ws_doubles;  // the sampler's per-warp scratch: the evaluator's plus two sweeps of draws
  bool exact;  // compiled for n_up = n_dn = NS
  const void *k_el, *k_psi, *k_metro, *k_expl, *k_el_deriv;
  const void *e_el, *e_psi, *e_metro, *e_expl, *e_el_deriv;
  const void *k_orb;  // orbital-parameter derivatives, kWarpsOrb warps per block
  const void *k_orb_small;  // the same with kWarpsOrbSmall warps (less shared memory)
  const void *k_nuc, *k_nuc_small;  // the same kernel in nuclear mode (qmc_nuclear_log_gradient)
  const void *k_orb_b, *k_orb_small_b, *k_nuc_b, *k_nuc_small_b;  // the four for a backflow wavefunction
  const void *x_orb, *x_orb_small, *x_nuc, *x_nuc_small;          // orbital_explicit_kernel for the groups those list
  const void *x_orb_b, *x_orb_small_b, *x_nuc_b, *x_nuc_small_b;
  int orb_ws_doubles;
  const void *k_frc, *k_frc_small;  // nuclear energy gradient (8 / 4 warps per block)
  const void *k_el_fuse, *e_el_fuse;   // E_L + fused eq. 6 reduction (without / with the e-e-n kernel)
  const void *b_psi, *b_metro, *b_el;  // backflow: values-only kernels, and the E_L kernel (explicit route)
  const void *be_psi, *be_metro;       // backflow values-only kernels with the e-e-n Jastrow kernel
  const void *b_tab;                   // backflow E_L from the reference's tables (F.6-F.9)
  const void *b_el_d, *b_tab_d;        // the same two with the parameter derivatives (eq. 6 factors, backflow weight last)
  const void *b_el_m, *b_tab_m, *b_el_dm, *b_tab_dm;  // the four with the many-body Jastrow kernels D.2 / D.3
  int bf_ws_doubles, bf_tab_ws_doubles, bf_e_doubles;
  int frc_ws_doubles;
};

template <int NS, int NMO, bool X>
Variant make_variant() {
  Variant v;
  v.NS = NS;
  v.NMO = NMO;
  v.LP = Geo<NS, NMO>::LP;
  v.exact = X;
  v.ws_doubles = Geo<NS, NMO>::total;
  v.wpb_psi_max = kWarpsPsiOf<NS>;
  v.psi_ws_doubles = Geo<NS, NMO>::totalC(true);
  v.metro_ws_doubles = Geo<NS, NMO>::totalC(true) + 2 * kDrawDoubles<NS>;
  v.k_el = (const void *)local_energy_kernel<NS, NMO, true, X, kWarpsEl>;
  v.k_psi = (const void *)local_energy_kernel<NS, NMO, false, X, kWarpsPsiOf<NS>>;
  v.k_metro = (const void *)metropolis_kernel<NS, NMO, X, kWarpsPsiOf<NS>>;
  v.k_expl = (const void *)explicit_energy_kernel<NS, NMO, X, kWarpsEl>;
  v.k_el_deriv = (const void *)local_energy_kernel<NS, NMO, true, X, kWarpsEl, true>;
  v.k_orb = (const void *)orbital_derivatives_kernel<NS, NMO, X, kWarpsOrb>;
  v.k_orb_small = (const void *)orbital_derivatives_kernel<NS, NMO, X, kWarpsOrbSmall>;
  v.k_nuc = (const void *)orbital_derivatives_kernel<NS, NMO, X, kWarpsOrb, true>;
  v.k_nuc_small = (const void *)orbital_derivatives_kernel<NS, NMO, X, kWarpsOrbSmall, true>;
  v.k_orb_b = (const void *)orbital_derivatives_kernel<NS, NMO, X, kWarpsOrb, false, true>;
  v.k_orb_small_b = (const void *)orbital_derivatives_kernel<NS, NMO, X, kWarpsOrbSmall, false, true>;
  v.k_nuc_b = (const void *)orbital_derivatives_kernel<NS, NMO, X, kWarpsOrb, true, true>;
  v.k_nuc_small_b = (const void *)orbital_derivatives_kernel<NS, NMO, X, kWarpsOrbSmall, true, true>;
  v.x_orb = (const void *)orbital_explicit_kernel<NS, NMO, X, kWarpsOrb>;
  v.x_orb_small = (const void *)orbital_explicit_kernel<NS, NMO, X, kWarpsOrbSmall>;
  v.x_nuc = (const void *)orbital_explicit_kernel<NS, NMO, X, kWarpsOrb, true>;
  v.x_nuc_small = (const void *)orbital_explicit_kernel<NS, NMO, X, kWarpsOrbSmall, true>;
  v.x_orb_b = (const void *)orbital_explicit_kernel<NS, NMO, X, kWarpsOrb, false, true>;
  v.x_orb_small_b = (const void *)orbital_explicit_kernel<NS, NMO, X, kWarpsOrbSmall, false, true>;
  v.x_nuc_b = (const void *)orbital_explicit_kernel<NS, NMO, X, kWarpsOrb, true, true>;
  v.x_nuc_small_b = (const void *)orbital_explicit_kernel<NS, NMO, X, kWarpsOrbSmall, true, true>;
  v.orb_ws_doubles = Geo<NS, NMO>::total + Geo<NS, NMO>::orbExtra;
  v.k_frc = (const void *)nuclear_energy_gradient_kernel<NS, NMO, X, 8>;
  v.k_frc_small = (const void *)nuclear_energy_gradient_kernel<NS, NMO, X, 4>;
  v.frc_ws_doubles = Geo<NS, NMO>::total + Geo<NS, NMO>::frcExtra;
  v.k_el_fuse = (const void *)local_energy_kernel<NS, NMO, true, X, kWarpsEl, true, false, false, true>;
  v.e_el_fuse = (const void *)local_energy_kernel<NS, NMO, true, X, kWarpsEl, true, true, false, true>;
  v.b_psi = (const void *)local_energy_kernel<NS, NMO, false, X, kWarpsPsiOf<NS>, false, false, true>;
  v.b_metro = (const void *)metropolis_kernel<NS, NMO, X, kWarpsPsiOf<NS>, false, true>;
  v.be_psi = (const void *)local_energy_kernel<NS, NMO, false, X, kWarpsPsiOf<NS>, false, true, true>;
  v.be_metro = (const void *)metropolis_kernel<NS, NMO, X, kWarpsPsiOf<NS>, true, true>;
  v.b_el = (const void *)backflow_energy_kernel<NS, NMO, kWarpsBfTab>;
  v.bf_ws_doubles = BfGeo<NS, NMO>::total;
  v.b_tab = (const void *)backflow_tables_kernel<NS, NMO, kWarpsBfTab>;
  v.b_el_d = (const void *)backflow_energy_kernel<NS, NMO, kWarpsBfTab, true>;
  v.b_tab_d = (const void *)backflow_tables_kernel<NS, NMO, kWarpsBfTab, true>;
  v.b_el_m = (const void *)backflow_energy_kernel<NS, NMO, kWarpsBfTab, false, true>;
  v.b_tab_m = (const void *)backflow_tables_kernel<NS, NMO, kWarpsBfTab, false, true>;
  v.b_el_dm = (const void *)backflow_energy_kernel<NS, NMO, kWarpsBfTab, true, true>;
  v.b_tab_dm = (const void *)backflow_tables_kernel<NS, NMO, kWarpsBfTab, true, true>;
  v.bf_tab_ws_doubles = BfGeoT<NS, NMO>::total;
  v.bf_e_doubles = BfGeoT<NS, NMO>::eDoubles;
  v.e_el = (const void *)local_energy_kernel<NS, NMO, true, X, kWarpsEl, false, true>;
  v.e_psi = (const void *)local_energy_kernel<NS, NMO, false, X, kWarpsPsiOf<NS>, false, true>;
  v.e_metro = (const void *)metropolis_kernel<NS, NMO, X, kWarpsPsiOf<NS>, true>;
  v.e_expl = (const void *)explicit_energy_kernel<NS, NMO, X, kWarpsEl, true>;
  v.e_el_deriv = (const void *)local_energy_kernel<NS, NMO, true, X, kWarpsEl, true, true>;
  return v;
}

}  // namespace qmc

#ifdef QMC_VARIANT_ARGS
// the body of a qmc_variant_*.cu:  QMC_VARIANT_NAME = function name, QMC_VARIANT_ARGS = NS, NMO, exact
namespace qmc {
Variant QMC_VARIANT_NAME() { return make_variant<QMC_VARIANT_ARGS>(); }
}  // namespace qmc
#endif
