// energy_tma.cuh -- the lattice sums behind pycool_energies as a TMA-fed z-march (sm_100a).   §8(a) row a7
//
// Per field f: sum pi_f^2, sum_x G[phi_f] (2.8), sum_x phi_f D[phi_f] (2.7); and sum_x V.
// Read-only pass over phi and pi: 2 sizeof(Real) bytes per field-site.  Same loading scheme as kick_tma (one
// (TX + 2G) x (TY + 2) x NF box of phi and of pi per z-plane into a ring of S shared-memory stages, halo included,
// ghost images making every box a plain in-bounds box), same register queue along z for the 27-point stencil.
//
// The gradient energy needs sum_x G[phi](x), G of (2.8).  G carries the centre value of the OUTPUT site in every term,
// so it does not decompose plane by plane; but the paper's own identity (2.17),
//     sum_x G[phi](x) = - sum_x phi(x) D[phi](x)        (summation by parts on the periodic lattice),
// does, and D annihilates constants (c0 = -(6c1 + 12c2 + 8c3)), so with psi = phi - ref, ref ONE value per field for
// the whole lattice (the field at site (0,0,0)): sum_x G[phi] = - sum_x psi D[psi], every term of which is of the size
// of the fluctuations -- no cancellation against the homogeneous part (the plain sum_x phi D[phi], kept as the third
// sum, loses ~6 digits on a preheating lattice).  One stencil, the kick's register queue, all arithmetic in double
// also for fp32 fields (reading G16).  The plain kernel (kernels.cuh: energy_sums) evaluates (2.8) term by term; the
// two agree to rounding (tested).
#pragma once
#include "kick_tma.cuh"

namespace pycool {

template <typename Real>
struct EnergyArgs {
  const Real* phi;        // the state arrays (for the lattice-wide reference value of each field)
  const Real* pi;
  const Scalars* sc;      // not NULL: the sums see phi' = phi + c_close pi (the pending closing half drift)
  double* partials;       // [3 NF + 1][nitems]
  Layout L;
  int zc;                 // planes per z-chunk
  int nbx, nby;           // x-y tiles; blockIdx.x = (bz nby + by) nbx + bx
  double c1, c2, c3;
  ModelParams mp;
};

template <typename Real, class Model, class T>
struct EnergySmem {
  using K = TmaSmem<Real, Model, T>;
  static constexpr size_t RED = (3 * Model::NF + 1) * (T::NT / 32) * sizeof(double);
  static constexpr size_t TOTAL = K::RAW + K::PSI + K::BARS + RED + 128;
};

template <typename Real, class Model, class T>
__global__ void __launch_bounds__(T::NT, T::MINB)
energy_tma(const __grid_constant__ CUtensorMap tm_phi, const __grid_constant__ CUtensorMap tm_pi,
           const EnergyArgs<Real> g) {
  using R2 = typename Vec2T<Real>::type;
  using SM = TmaSmem<Real, Model, T>;
  constexpr int NF = Model::NF, NQ = 3 * NF + 1, TX = T::TX, TY = T::TY, S = T::S, G = T::G, PX = T::PX;
  constexpr int NT = T::NT, J = T::J, PLANE = T::PLANE;

  extern __shared__ unsigned char smem_dyn[];
  unsigned char* base = smem_dyn + ((128u - (smem_addr(smem_dyn) & 127u)) & 127u);
  unsigned char* raw = base;                                   // [S][2][BOXA]
  Real* psi = reinterpret_cast<Real*>(base + SM::RAW);         // [2][BOXA]
  const uint32_t bars = smem_addr(base + SM::RAW + SM::PSI);
  double* red = reinterpret_cast<double*>(base + SM::RAW + SM::PSI + SM::BARS);

  const Layout& L = g.L;
  const int N = L.N;
  const int tid = threadIdx.x;
  const int tx2 = tid % (TX / 2), tyj = tid / (TX / 2);
  constexpr int NB_RUN = 128 / (2 * (int)sizeof(Real));        // neighbour loads, every other run of threads swapped:
  const bool nb_swap = ((tx2 / NB_RUN) & 1) != 0;              // no bank conflict (kick_tma.cuh: march_item)
  const int nb_first = nb_swap ? 2 : -1, nb_second = nb_swap ? -1 : 2;
  const int item = blockIdx.x, nbxy = g.nbx * g.nby;
  const int bz = item / nbxy, r_ = item - bz * nbxy, by = r_ / g.nbx;
  const int x0 = (r_ - by * g.nbx) * TX, y0 = by * TY, z0 = bz * g.zc;
  const int nz = min(g.zc, N - z0);
  const int nload = nz + 2;                                    // planes z0-1 .. z0+nz

  auto issue = [&](int i) {                                    // load index i <-> plane p = i - 1 (thread 0)
    const int s = i % S;
    const uint32_t bar = bars + 8u * s;
    const uint32_t dst = smem_addr(raw + (size_t)s * 2 * SM::BOXA);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(bar, (uint32_t)(2 * SM::BOX));
    int gz = z0 + i - 1;
    gz = gz < 0 ? gz + N : (gz >= N ? gz - N : gz);
    tma_load_4d(dst, &tm_phi, bar, x0, y0, gz, 0);
    tma_load_4d(dst + (uint32_t)SM::BOXA, &tm_pi, bar, x0, y0, gz, 0);
  };
  if (tid == 0) {
    for (int s = 0; s < S; ++s) mbar_init(bars + 8u * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    for (int i = 0; i < S && i < nload; ++i) issue(i);
  }

  const double c1 = g.c1, c2 = g.c2, c3 = g.c3;
  const double c0 = -(6.0 * c1 + 12.0 * c2 + 8.0 * c3);
  const bool drift = g.sc != nullptr;                          // block-uniform
  const Real cd = drift ? Real(g.sc->c_close) : Real(0);
  const typename Model::template Coef<double> coef(g.mp);

  bool valid[J];
  {
    const int gx = x0 + 2 * tx2;
#pragma unroll
    for (int j = 0; j < J; ++j) valid[j] = gx < N && y0 + J * tyj + j < N;
  }
  const int own_sm = (J * tyj + 1) * PX + G + 2 * tx2;
  constexpr int NHT = (T::NHP + NT - 1) / NT;
  int halo_sm[NHT];
  halo_pairs_of_thread<T>(tid, halo_sm);

  // per site: value pair of plane p-1 (phi, pi), accumulators of D[psi] (A, B)
  double2 pphi[NF][J], ppi[NF][J], A[NF][J], B[NF][J];
  Real ref[NF];
  double acc[NQ];
#pragma unroll
  for (int q = 0; q < NQ; ++q) acc[q] = 0.0;
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    // one reference value per field for the WHOLE lattice: the field at site (0,0,0) as a flushed state holds it.
    // fp32 fields: psi is stored in shared memory as a float, and phi - ref is exact in float only next to ref
    // (a mean-zero field would pick up 6e-8 relative per site, which D does not annihilate), so no reference is
    // subtracted: the stencil runs in double on the exact float values (loses 5 of 16 digits, far below fp32).
    const size_t o0 = L.at(f, 0, 0, 0);
    if constexpr (sizeof(Real) == 4) ref[f] = Real(0);
    else ref[f] = drift ? fma(cd, g.pi[o0], g.phi[o0]) : g.phi[o0];
#pragma unroll
    for (int j = 0; j < J; ++j) pphi[f][j] = ppi[f][j] = A[f][j] = B[f][j] = double2{0.0, 0.0};
  }

  __syncthreads();                                             // barriers initialised before anyone waits

#pragma unroll 1
  for (int p = -1; p <= nz; ++p) {
    const int i = p + 1, s = i % S;
    const Real* rphi = reinterpret_cast<const Real*>(raw + (size_t)s * 2 * SM::BOXA);
    const Real* rpi = reinterpret_cast<const Real*>(raw + (size_t)s * 2 * SM::BOXA + SM::BOXA);
    Real* pb = psi + (size_t)(i & 1) * (SM::BOXA / sizeof(Real));
    mbar_wait(bars + 8u * s, (uint32_t)((i / S) & 1));

    // ---- 1. psi = phi - ref into shared memory (own pairs and halo ring); keep phi, pi of the own sites
    double2 cphi[NF][J], cpi[NF][J];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
#pragma unroll
      for (int j = 0; j < J; ++j) {
        const int o = f * PLANE + own_sm + j * PX;
        R2 a = *reinterpret_cast<const R2*>(rphi + o);
        const R2 b = *reinterpret_cast<const R2*>(rpi + o);
        if (drift) { a.x = fma(cd, b.x, a.x); a.y = fma(cd, b.y, a.y); }     // as drift_flush would store it
        cphi[f][j] = double2{(double)a.x, (double)a.y};
        cpi[f][j] = double2{(double)b.x, (double)b.y};
        *reinterpret_cast<R2*>(pb + o) = R2{a.x - ref[f], a.y - ref[f]};
      }
#pragma unroll
      for (int k = 0; k < NHT; ++k)
        if (halo_sm[k] >= 0) {
          const int o = f * PLANE + halo_sm[k];
          R2 a = *reinterpret_cast<const R2*>(rphi + o);
          if (drift) {
            const R2 b = *reinterpret_cast<const R2*>(rpi + o);
            a.x = fma(cd, b.x, a.x); a.y = fma(cd, b.y, a.y);
          }
          *reinterpret_cast<R2*>(pb + o) = R2{a.x - ref[f], a.y - ref[f]};
        }
    }
    __syncthreads();                                           // psi plane complete; raw stage s consumed
    if (tid == 0 && i + S < nload) issue(i + S);

    // ---- 2. in-plane sums of psi and psi^2 for plane p; 3. finalise plane p-1
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const Real* sp = pb + f * PLANE + own_sm - PX;           // row above the first own row
      double Rx[J + 2], Cx[J + 2], Ry[J + 2], Cy[J + 2];       // psi: side sums and centres of x-outputs 0, 1
#pragma unroll
      for (int r = 0; r < J + 2; ++r) {
        const Real n0 = sp[r * PX + nb_first], n1 = sp[r * PX + nb_second];   // bank-conflict-free order: kick_tma.cuh
        double mx, my;
        if (r >= 1 && r <= J) {                                // an own row: what this thread stored, from its registers
          mx = (double)(Real(cphi[f][r - 1].x) - ref[f]); my = (double)(Real(cphi[f][r - 1].y) - ref[f]);
        } else {
          const R2 m = *reinterpret_cast<const R2*>(sp + r * PX);
          mx = (double)m.x; my = (double)m.y;
        }
        const double l = (double)(nb_swap ? n1 : n0), rr = (double)(nb_swap ? n0 : n1);
        Rx[r] = l + my; Cx[r] = mx; Ry[r] = mx + rr; Cy[r] = my;
      }
#pragma unroll
      for (int j = 0; j < J; ++j) {
        double Dx, Dy;
        {
          const double P0 = Cx[j + 1], P1 = Rx[j + 1] + (Cx[j] + Cx[j + 2]), P2 = Rx[j] + Rx[j + 2];
          const double up = fma(c3, P2, fma(c2, P1, c1 * P0));
          Dx = A[f][j].x + up;
          A[f][j].x = fma(c2, P2, fma(c1, P1, fma(c0, P0, B[f][j].x)));
          B[f][j].x = up;
        }
        {
          const double P0 = Cy[j + 1], P1 = Ry[j + 1] + (Cy[j] + Cy[j + 2]), P2 = Ry[j] + Ry[j + 2];
          const double up = fma(c3, P2, fma(c2, P1, c1 * P0));
          Dy = A[f][j].y + up;
          A[f][j].y = fma(c2, P2, fma(c1, P1, fma(c0, P0, B[f][j].y)));
          B[f][j].y = up;
        }
        if (p >= 1 && valid[j]) {                              // output plane p-1 (an own plane: 0 .. nz-1)
          const double rf = (double)ref[f];
          const double px = pphi[f][j].x, py = pphi[f][j].y;   // phi
          const double sx = px - rf, sy = py - rf;             // psi
          acc[3 * f] = fma(ppi[f][j].x, ppi[f][j].x, fma(ppi[f][j].y, ppi[f][j].y, acc[3 * f]));
          acc[3 * f + 1] = fma(-sx, Dx, fma(-sy, Dy, acc[3 * f + 1]));     // sum G = - sum psi D[psi]   (2.17)
          acc[3 * f + 2] = fma(px, Dx, fma(py, Dy, acc[3 * f + 2]));       // sum phi D[phi] as written
        }
      }
    }
    if (p >= 1) {
#pragma unroll
      for (int j = 0; j < J; ++j)
        if (valid[j]) {
          double ph[NF], dV[NF];
#pragma unroll
          for (int f = 0; f < NF; ++f) ph[f] = pphi[f][j].x;
          acc[3 * NF] += Model::template eval<double>(coef, ph, dV);
#pragma unroll
          for (int f = 0; f < NF; ++f) ph[f] = pphi[f][j].y;
          acc[3 * NF] += Model::template eval<double>(coef, ph, dV);
        }
    }
#pragma unroll
    for (int f = 0; f < NF; ++f)
#pragma unroll
      for (int j = 0; j < J; ++j) { pphi[f][j] = cphi[f][j]; ppi[f][j] = cpi[f][j]; }
  }

  block_reduce<NQ, NT>(acc, red);
  if (tid == 0) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) g.partials[(size_t)q * gridDim.x + item] = acc[q];
  }
}

}  // namespace pycool
