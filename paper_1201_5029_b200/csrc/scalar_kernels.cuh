// scalar_kernels.cuh -- the small non-template kernels of the library: stand-alone scalar update, row reduction,
// scalar stores.  Included by pycool.cu only (non-template __global__ functions must have one definition).
#pragma once
#include "kernels.cuh"

namespace pycool {

// Stand-alone form: reduces partials [3][nblocks] (mode 1) and advances the scalars.  Used for the opening of a
// call (mode 0) and when the fused tail is switched off.
__global__ void __launch_bounds__(kReduceThreads)
scalar_update(Scalars* __restrict__ sc, const double* __restrict__ partials, int nblocks, ScalarConst k,
              StageLen len, int mode) {
  __shared__ double sh[kReduceThreads];
  double SD = 0, SV = 0, SP = 0;
  if (mode == 1) {
    SD = block_sum_fixed<kReduceThreads>(partials, nblocks, sh);
    SV = block_sum_fixed<kReduceThreads>(partials + nblocks, nblocks, sh);
    SP = block_sum_fixed<kReduceThreads>(partials + 2 * (size_t)nblocks, nblocks, sh);
  }
  if (threadIdx.x != 0) return;
  Scalars s = *sc;
  scalar_advance(s, k, len, mode, SD, SV, SP);
  *sc = s;
}

// out[q] = fixed-order sum of partials[q][0..nb);  grid = nq blocks
__global__ void __launch_bounds__(kReduceThreads) reduce_rows(const double* __restrict__ partials, int nb,
                                                             double* __restrict__ out) {
  __shared__ double sh[kReduceThreads];
  const double r = block_sum_fixed<kReduceThreads>(partials + (size_t)blockIdx.x * nb, nb, sh);
  if (threadIdx.x == 0) out[blockIdx.x] = r;
}

__global__ void store_spi2(Scalars* sc, const double* v) {
  sc->Spi2 = *v;
  if (!isfinite(*v)) sc->nonfinite = 1;
}
__global__ void set_scalars(Scalars* sc, double a, double p_a, int set_pa) {
  sc->a = a; sc->a_sync = a;
  if (set_pa) { sc->p_a = p_a; sc->pa_sync = p_a; }
  sc->c_close = 0.0;
}

// The energy read-out finished on the device: adds the per-block partial sums of an energy launch
// ([3 nf + 1][nb]: per field sum pi^2, sum G, sum phi D phi; then sum V) in index order and forms the lattice
// averages, rho, P (2.16) + (2.20), H (2.14) and the residual (3.1) at the time-synchronised scale factor
// (Scalars::a_sync) -- one entry of the energy log, or the answer of pycool_energies.  Separate IEEE operations
// in a fixed order (no FMA contraction), so the same sums give the same entry bit for bit wherever it is computed.
struct EnergyConst {
  double V, dx2, mpl, rho_g, rho_m;   // V_L, dx^2, reduced Planck mass (+INF: static), (2.20) densities
  int nf;
};
__global__ void __launch_bounds__(kReduceThreads)
energy_finish(const double* __restrict__ partials, int nb, Scalars* __restrict__ sc, EnergyConst k,
              pycool_energy* __restrict__ out) {
  __shared__ double sh[kReduceThreads];
  __shared__ double s[16];
  const int nq = 3 * k.nf + 1;
  for (int q = 0; q < nq; ++q) {
    const double r = block_sum_fixed<kReduceThreads>(partials + (size_t)q * nb, nb, sh);
    if (threadIdx.x == 0) s[q] = r;
  }
  if (threadIdx.x != 0) return;
  const double a = sc->a_sync, p_a = sc->pa_sync;
  const double a2 = __dmul_rn(a, a), a4 = __dmul_rn(a2, a2), a6 = __dmul_rn(a4, a2);
  const double dK = __dmul_rn(__dmul_rn(2.0, a6), k.V);                     // 2 a^6 V_L
  const double dG = __dmul_rn(__dmul_rn(__dmul_rn(2.0, a2), k.dx2), k.V);   // 2 a^2 dx^2 V_L
  pycool_energy e;
  for (int f = 0; f < 4; ++f) e.kin[f] = e.grad[f] = e.sum_phiDphi[f] = 0.0;
  const double Vbar = __ddiv_rn(s[3 * k.nf], k.V);
  double rho = __dadd_rn(__dadd_rn(Vbar, __ddiv_rn(k.rho_g, a4)), __ddiv_rn(k.rho_m, __dmul_rn(a2, a)));
  double P = __dadd_rn(-Vbar, __ddiv_rn(k.rho_g, __dmul_rn(__dmul_rn(3.0, a2), a2)));
  bool finite = isfinite(s[3 * k.nf]);
  for (int f = 0; f < k.nf; ++f) {
    const double K = __ddiv_rn(s[3 * f], dK), Gr = __ddiv_rn(s[3 * f + 1], dG);
    e.kin[f] = K; e.grad[f] = Gr; e.sum_phiDphi[f] = -__ddiv_rn(s[3 * f + 2], dG);
    rho = __dadd_rn(rho, __dadd_rn(K, Gr));
    P = __dadd_rn(P, __dsub_rn(K, __ddiv_rn(Gr, 3.0)));
    finite = finite && isfinite(s[3 * f]) && isfinite(s[3 * f + 1]) && isfinite(s[3 * f + 2]);
  }
  if (!finite) sc->nonfinite = 1;
  const double ap = -__ddiv_rn(p_a, __dmul_rn(__dmul_rn(__dmul_rn(6.0, k.V), k.mpl), k.mpl));  // (2.14)
  const double H = __ddiv_rn(ap, a2);
  e.a = a; e.p_a = p_a; e.eta = sc->eta;
  e.pot = Vbar; e.rho = rho; e.pressure = P; e.hubble = H;
  const double den = __dmul_rn(__dmul_rn(__dmul_rn(__dmul_rn(3.0, k.mpl), k.mpl), H), H);
  e.residual = isinf(k.mpl) ? 0.0 : fabs(__dsub_rn(__ddiv_rn(rho, den), 1.0));                 // (3.1)
  *out = e;
}

}  // namespace pycool
