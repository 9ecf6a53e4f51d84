// linear.cuh -- sm_100a kernels of the linearised solver (arXiv 1201.5029 section 2.2, (2.35)-(2.38), (2.49)-(2.51)).
//
//   lin_background   one thread: the background (a, p_a, phi_0, pi_0) through every stage of the call -- flows H1, H2,
//                    H3 of (2.49) in the order (2.50) -- writing, per stage, the three coefficients the perturbation
//                    flows H4, H5 need: e/a^2, a^2 h/dx^2 and a^4 h V_ij(phi_0).
//   lin_growth       one thread per (distinct k_eff^2 class, column of M): the growth function M(tau, k_eff^2) 1_c of
//                    (2.51) through every stage, coefficients staged through shared memory.
//   lin_apply        one thread per Fourier mode of the half spectrum: mode <- M(class of the mode) mode.
//   lin_naive        one thread per Fourier mode: the mode itself through every stage (the paper's "naive version").
//   lin_background_energy, lin_set_pa, lin_zero_mode, lin_scale   small helpers.
//
// The paper evolves the background redundantly in the first thread of every block so that blocks need
// not synchronise; here it is evolved once, ahead of the growth kernel, and its per-stage coefficients are a table
// (a few KB) that every block streams through shared memory -- the growth kernel's inner loop is then pure fp64 FMA
// work on registers, bound by the fp64 pipe.
#pragma once
#include <cfloat>
#include <cmath>
#include <cstddef>

namespace pycool {

constexpr int kLinMaxNF = 4;

struct LinBackground {      // device-resident
  double a, p_a, eta;
  double phi0[kLinMaxNF], pi0[kLinMaxNF];
};

struct LinConst {
  int model, nf;
  double p[8];
  double inv_mpl2;          // 0 for a static background
  double den;               // 6 V_L mpl^2 (+INF: static)
  double VL, rho_g, rho_m, mpl;
  double dx2;
  double c[4];              // stencil c0..c3
};

// Per-stage coefficients of the perturbation flows, in the order they are used: H4(e), H5(h), H4(e).
template <int NF>
struct LinStage {
  double c4;                // e / a^2                  dPhi += c4 dPi                                   H4, (2.38)
  double kD;                // a^2 h / dx^2             dPi_i -= kD k_eff^2 dPhi_i                       H5
  double Hh[NF * NF];       // a^4 h V_ij(phi_0)        dPi_i -= sum_j Hh_ij dPhi_j                      H5, (2.26)
};

// V, dV/dphi_i and V_ij at a homogeneous point.  (3.2) PAPER.md:427, (3.3) PAPER.md:456, (3.4) PAPER.md:481 with the
// readings G6-G8; the second derivatives are what (2.26)/(2.27) need and the paper prints for (3.2) only.
__device__ inline double lin_potential(const LinConst& k, const double* phi, double* dV, double* H) {
  const int nf = k.nf;
  for (int i = 0; i < nf * nf; ++i) H[i] = 0.0;
  double V = 0.0;
  switch (k.model) {
    case 0:                                                    // free: sum 1/2 m_f^2 phi_f^2
      for (int f = 0; f < nf; ++f) {
        dV[f] = k.p[f] * phi[f];
        V += 0.5 * dV[f] * phi[f];
        H[f * nf + f] = k.p[f];
      }
      break;
    case 1: {                                                  // chaotic: 1/2 m^2 phi^2 + 1/2 g^2 phi^2 chi^2
      const double m2 = k.p[0], g2 = k.p[1], ph = phi[0], ch = phi[1];
      V = 0.5 * m2 * ph * ph + 0.5 * g2 * ph * ph * ch * ch;
      dV[0] = m2 * ph + g2 * ph * ch * ch;
      dV[1] = g2 * ph * ph * ch;
      H[0] = m2 + g2 * ch * ch;                                // (2.27)
      H[1] = H[2] = 2.0 * g2 * ph * ch;
      H[3] = g2 * ph * ph;
      break;
    }
    case 2: {                                                  // oscillon: 1/2 m^2 phi^2 - lambda/4 phi^4 + g6/6 phi^6
      const double m2 = k.p[0], lam = k.p[1], g6 = k.p[2], ph = phi[0], p2 = ph * ph;
      V = 0.5 * m2 * p2 - lam / 4.0 * p2 * p2 + g6 / 6.0 * p2 * p2 * p2;
      dV[0] = m2 * ph - lam * p2 * ph + g6 * p2 * p2 * ph;
      H[0] = m2 - 3.0 * lam * p2 + 5.0 * g6 * p2 * p2;
      break;
    }
    default: {                                                 // Q-ball: m^2 r2 (1 + K ln(r2/M^2)) + six r2^3
      const double m2 = k.p[0], K = k.p[1], M2 = k.p[2], six = k.p[3] * k.inv_mpl2;
      const double r2 = 0.5 * (phi[0] * phi[0] + phi[1] * phi[1]);
      const bool tiny = r2 < DBL_MIN;                          // reading G8
      const double lg = tiny ? 0.0 : log(r2 / M2);
      const double common = m2 * (1.0 + K + K * lg) + 3.0 * six * r2 * r2;
      V = m2 * r2 * (1.0 + K * lg) + six * r2 * r2 * r2;
      dV[0] = common * phi[0];
      dV[1] = common * phi[1];
      const double dc = tiny ? 0.0 : m2 * K / r2 + 6.0 * six * r2;   // d common / d r2, and d r2 / d phi_j = phi_j
      for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) H[i * 2 + j] = (i == j ? common : 0.0) + dc * phi[i] * phi[j];
      break;
    }
  }
  return V;
}

// The background through nsteps x nstages stages; table[s] = coefficients of stage s for the perturbations.
// One thread (launch <<<1, 1>>>): the recurrence is serial, so what matters is the length of its dependent chain.
// Within one stage of (2.50), H1 H2 H3 [H4 H5 H4] H3 H2 H1, the scale factor changes only in H1 and phi_0 only in H2:
// both H2 halves and both H3 halves see the same a, and both H3 halves and the perturbation flows the same phi_0 --
// one reciprocal of a and one evaluation of the potential serve the whole stage.
template <int NF>
__global__ void lin_background(LinBackground* bg, const LinConst k, const double* __restrict__ w, int nstages,
                               int nsteps, double dt, LinStage<NF>* __restrict__ table) {
  LinBackground b = *bg;
  const double inv_den = 1.0 / k.den, Vrho_m = k.VL * k.rho_m;
  size_t idx = 0;
  for (int n = 0; n < nsteps; ++n) {
    for (int s = 0; s < nstages; ++s, ++idx) {
      const double h = w[s] * dt, e = 0.5 * h;
      b.a -= b.p_a * inv_den * e;                                                 // H1(e)        (2.35)
      const double a = b.a, a2 = a * a, a3 = a2 * a, a4 = a2 * a2;
      const double ia = 1.0 / a, ia2 = ia * ia, ia3 = ia2 * ia;
      double sp = 0.0;
      for (int f = 0; f < NF; ++f) sp += b.pi0[f] * b.pi0[f];
      b.p_a += (k.VL * sp * ia3 - Vrho_m) * e;                                    // H2(e)        (2.35), (2.20)
      for (int f = 0; f < NF; ++f) b.phi0[f] += b.pi0[f] * ia2 * e;               //              (2.36)
      double dV[kLinMaxNF], H[kLinMaxNF * kLinMaxNF];
      const double V = lin_potential(k, b.phi0, dV, H);
      const double dpa = -4.0 * a3 * k.VL * V * e;
      b.p_a += dpa;                                                               // H3(e)        (2.35)
      for (int f = 0; f < NF; ++f) b.pi0[f] -= a4 * dV[f] * e;                    //              (2.36)
      LinStage<NF> st;                                                            // H4(e) H5(h) H4(e) see this a, phi_0
      st.c4 = e * ia2;
      st.kD = a2 / k.dx2 * h;
      for (int i = 0; i < NF * NF; ++i) st.Hh[i] = a4 * H[i] * h;
      table[idx] = st;
      b.p_a += dpa;                                                               // H3(e)
      for (int f = 0; f < NF; ++f) b.pi0[f] -= a4 * dV[f] * e;
      sp = 0.0;
      for (int f = 0; f < NF; ++f) sp += b.pi0[f] * b.pi0[f];
      b.p_a += (k.VL * sp * ia3 - Vrho_m) * e;                                    // H2(e)
      for (int f = 0; f < NF; ++f) b.phi0[f] += b.pi0[f] * ia2 * e;
      b.a -= b.p_a * inv_den * e;                                                 // H1(e)
    }
    b.eta += dt;
  }
  *bg = b;
}

// p_a from the first Friedmann equation (2.18) on the background alone, expanding branch (reading G10).
__global__ void lin_set_pa(LinBackground* bg, const LinConst k) {
  LinBackground b = *bg;
  double dV[kLinMaxNF], H[kLinMaxNF * kLinMaxNF];
  const double V = lin_potential(k, b.phi0, dV, H);
  const double a2 = b.a * b.a;
  double s = 0.0;
  for (int f = 0; f < k.nf; ++f) s += b.pi0[f] * b.pi0[f];
  const double rho = s / (2.0 * a2 * a2 * a2) + V + k.rho_g / (a2 * a2) + k.rho_m / (a2 * b.a);
  bg->p_a = -6.0 * k.VL * k.mpl * a2 * sqrt(rho / 3.0);
}

struct LinEnergyOut { double kin, pot, rho, hubble, residual; };
__global__ void lin_background_energy(const LinBackground* bg, const LinConst k, LinEnergyOut* out) {
  const LinBackground b = *bg;
  double dV[kLinMaxNF], H[kLinMaxNF * kLinMaxNF];
  const double V = lin_potential(k, b.phi0, dV, H);
  const double a2 = b.a * b.a;
  double s = 0.0;
  for (int f = 0; f < k.nf; ++f) s += b.pi0[f] * b.pi0[f];
  LinEnergyOut o;
  o.kin = s / (2.0 * a2 * a2 * a2);
  o.pot = V;
  o.rho = o.kin + V + k.rho_g / (a2 * a2) + k.rho_m / (a2 * b.a);
  const double ap = -b.p_a / k.den;
  o.hubble = ap / a2;
  o.residual = (k.inv_mpl2 > 0.0 && o.hubble != 0.0) ? fabs(o.rho * k.inv_mpl2 / (3.0 * o.hubble * o.hubble) - 1.0) : 0.0;
  *out = o;
}

// ------------------------------------------------------------------------------------------------ classes (G28)
// k_eff^2(n) is a symmetric function of (cos 2 pi n_x/N, cos 2 pi n_y/N, cos 2 pi n_z/N), so modes with the same
// sorted triple lo <= mid <= hi of |n_i| (0 .. M = floor(N/2)) share one growth matrix.  Classes are numbered in
// the order (hi, mid, lo): rank = hi(hi+1)(hi+2)/6 + mid(mid+1)/2 + lo (combinatorial number system).
__host__ __device__ __forceinline__ unsigned long long lin_tet(unsigned long long h) { return h * (h + 1) * (h + 2) / 6; }
__host__ __device__ __forceinline__ unsigned long long lin_tri(unsigned long long m) { return m * (m + 1) / 2; }

__device__ __forceinline__ unsigned lin_class_of(int a, int b, int c) {   // any order, each 0 .. M
  int lo = min(a, min(b, c)), hi = max(a, max(b, c)), mid = a + b + c - lo - hi;
  return (unsigned)(lin_tet((unsigned)hi) + lin_tri((unsigned)mid) + (unsigned)lo);
}
__device__ __forceinline__ void lin_class_triple(unsigned t, int& lo, int& mid, int& hi) {
  int h = (int)__powf(6.0f * (float)t + 1.0f, 0.33333334f);   // a guess within a few units; corrected below
  while (lin_tet((unsigned)h + 1) <= t) ++h;
  while (h > 0 && lin_tet((unsigned)h) > t) --h;
  const unsigned rem = t - (unsigned)lin_tet((unsigned)h);
  int m = (int)((sqrtf(8.0f * (float)rem + 1.0f) - 1.0f) * 0.5f);
  while (lin_tri((unsigned)m + 1) <= rem) ++m;
  while (m > 0 && lin_tri((unsigned)m) > rem) --m;
  hi = h; mid = m; lo = (int)(rem - (unsigned)lin_tri((unsigned)m));
}
// minus the eigenvalue of the stencil (2.7) on the plane wave with integer wave vector (n1, n2, n3)
__device__ __forceinline__ double lin_k_eff2(const double (&c)[4], int N, int n1, int n2, int n3) {
  const double s = 2.0 / (double)N;
  const double C1 = cospi(s * n1), C2 = cospi(s * n2), C3 = cospi(s * n3);
  return -(c[0] + 2.0 * c[1] * (C1 + C2 + C3) + 4.0 * c[2] * (C1 * C2 + C2 * C3 + C3 * C1) + 8.0 * c[3] * C1 * C2 * C3);
}

struct LinStencil { double c[4]; };

constexpr int kLinChunk = 64;        // stages staged through shared memory at a time
constexpr int kLinThreads = 256;

// One stage of the perturbation flows H4(e) H5(h) H4(e) of (2.50) on NF (phi, pi) pairs with one k_eff^2.
template <int NF>
__device__ __forceinline__ void lin_stage(const double* __restrict__ st /* LinStage<NF> as doubles */, double k2,
                                          double (&phi)[NF], double (&pi)[NF]) {
  const double c4 = st[0], kk = st[1] * k2;
#pragma unroll
  for (int i = 0; i < NF; ++i) phi[i] = fma(c4, pi[i], phi[i]);
  double npi[NF];                                              // H5 reads the phi of before the kick: all fields first
#pragma unroll
  for (int i = 0; i < NF; ++i) {
    npi[i] = fma(-kk, phi[i], pi[i]);
#pragma unroll
    for (int j = 0; j < NF; ++j) npi[i] = fma(-st[2 + i * NF + j], phi[j], npi[i]);
  }
#pragma unroll
  for (int i = 0; i < NF; ++i) pi[i] = npi[i];
#pragma unroll
  for (int i = 0; i < NF; ++i) phi[i] = fma(c4, pi[i], phi[i]);
}

// Block-wide copy of stages [base, base + n) of the table into shared memory.
template <int NF>
__device__ __forceinline__ void lin_stage_chunk(const LinStage<NF>* __restrict__ table, size_t base, int n, double* sh) {
  constexpr int W = 2 + NF * NF;
  const double* src = reinterpret_cast<const double*>(table + base);
  for (int i = threadIdx.x; i < n * W; i += blockDim.x) sh[i] = src[i];
}

// Growth functions (2.51): thread g = class * 2 NF + column integrates M(tau, k_eff^2) 1_column through all
// `nst` stages and writes column `column` of the class's matrix, M[class][row][column], rows (dPhi_1, dPi_1, ..).
template <int NF>
__global__ void __launch_bounds__(kLinThreads)
lin_growth(const LinStage<NF>* __restrict__ table, size_t nst, LinStencil sc, int N, unsigned nclasses,
           double* __restrict__ M) {
  constexpr int W = 2 + NF * NF, C = 2 * NF;
  __shared__ double sh[kLinChunk * W];
  const unsigned g = blockIdx.x * blockDim.x + threadIdx.x;    // < classes x 2 NF <= 1.5e9 at N = 2048
  const unsigned t = g / C;
  const int col = (int)(g - t * C);
  const bool live = t < nclasses;
  double k2 = 0.0;
  if (live) {
    int lo, mid, hi;
    lin_class_triple(t, lo, mid, hi);
    k2 = lin_k_eff2(sc.c, N, lo, mid, hi);
  }
  double phi[NF], pi[NF];
#pragma unroll
  for (int i = 0; i < NF; ++i) {
    phi[i] = (col == 2 * i) ? 1.0 : 0.0;
    pi[i] = (col == 2 * i + 1) ? 1.0 : 0.0;
  }
  for (size_t base = 0; base < nst; base += kLinChunk) {
    const int n = (int)min((size_t)kLinChunk, nst - base);
    __syncthreads();
    lin_stage_chunk<NF>(table, base, n, sh);
    __syncthreads();
    if (live)
      for (int s = 0; s < n; ++s) lin_stage<NF>(sh + s * W, k2, phi, pi);
  }
  if (live) {
    double* m = M + (size_t)t * C * C + col;
#pragma unroll
    for (int i = 0; i < NF; ++i) {
      m[(2 * i) * C] = phi[i];
      m[(2 * i + 1) * C] = pi[i];
    }
  }
}

// Mode kernels run on a 2-D grid: blockIdx.y = iz, and blockIdx.x * blockDim.x + threadIdx.x = iy (N/2 + 1) + ix
// inside the plane (32-bit arithmetic; one division per thread).  Modes: [iz][iy][ix], ix = 0 .. N/2.
// Returns false for a thread beyond the plane; m = linear mode index, (ax, ay, az) = folded wave numbers.
__device__ __forceinline__ bool lin_mode_of_thread(int N, size_t& m, int& ax, int& ay, int& az) {
  const unsigned nxh = (unsigned)N / 2 + 1, plane = (unsigned)N * nxh;
  const unsigned q = blockIdx.x * blockDim.x + threadIdx.x;
  const int iz = (int)blockIdx.y;
  const unsigned iy = q / nxh;
  ax = (int)(q - iy * nxh); ay = min((int)iy, N - (int)iy); az = min(iz, N - iz);
  m = (size_t)iz * plane + q;
  return q < plane;
}

// mode <- M(class of the mode) mode   (2.51).  dPhi, dPi: [NF][nmodes] complex.
// The matrices are a gather: neighbouring modes belong to different classes.  One thread per (mode, R rows of M),
// R = kLinApplyRows = 2: the NF threads of a mode read the 2 NF rows of its matrix -- together one contiguous
// (2 NF)^2 x 8 bytes, a whole line at NF = 2, in 256-bit loads -- and each the mode's 2 NF complex values (the same
// addresses within the group: broadcast), and write the field's (dPhi, dPi) pair.  No shared memory, no shuffles.
// The kernel is bound by L1 wavefronts, not by bytes in flight: a 16-byte load costs a wavefront per quarter warp
// however many of its threads share an address, so what counts is how many modes a quarter warp covers -- R = 1 (a
// thread per row; two 16-byte loads per row) ran at 0.66 of the HBM roofline at 256^3, with 256-bit row loads 0.75,
// R = 2 0.86, R = 2 NF (a thread per mode, its matrix in strided loads) 0.80; earlier forms: thread per mode with
// 16-byte matrix loads 0.57 (L1 95 % busy), matrices staged through shared memory 0.63, several modes per thread
// 0.52-0.56.  The update is in place, so the block synchronises between its reads and its writes.
constexpr int kLinApplyRows = 2;

// One row of a growth matrix, 2 NF doubles, read-only path.  Even NF: rows are 32-byte aligned (the table is, and a
// row is 32 or 64 bytes), so a row moves in 256-bit loads (LDG.E.256, sm_100): the four threads of a mode at NF = 2
// then fetch its whole 128-byte matrix in ONE instruction -- one L1 wavefront per mode where two 16-byte loads took two.
template <int NF>
__device__ __forceinline__ void lin_load_row(const double2* __restrict__ row, double2 (&mm)[NF]) {
  if constexpr (NF % 2 == 0) {
#pragma unroll
    for (int c = 0; c < NF; c += 2)
      asm("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];"
          : "=d"(mm[c].x), "=d"(mm[c].y), "=d"(mm[c + 1].x), "=d"(mm[c + 1].y)
          : "l"(row + c));
  } else {
#pragma unroll
    for (int c = 0; c < NF; ++c) mm[c] = __ldg(row + c);
  }
}

template <int NF, int R> struct LinApplyCfg {
  static constexpr int C = 2 * NF;                            // rows of M
  static_assert(C % R == 0, "rows per thread divide the rows of M");
  static constexpr int TPM = C / R;                           // threads per mode
  static constexpr int NT = 256;
  static constexpr int MPB = NT / TPM;                        // modes per block (NF = 3, R = 2: 85, one thread idle)
};
template <int NF, int R>
__global__ void __launch_bounds__(LinApplyCfg<NF, R>::NT)
lin_apply(double2* __restrict__ dPhi, double2* __restrict__ dPi, const double* __restrict__ M, int N, size_t nmodes) {
  using K = LinApplyCfg<NF, R>;
  constexpr int C = K::C, TPM = K::TPM;
  const unsigned nxh = (unsigned)N / 2 + 1, plane = (unsigned)N * nxh;
  const unsigned ml = threadIdx.x / TPM, rp = threadIdx.x - ml * TPM;   // mode of the block, row group of the mode
  const unsigned q = blockIdx.x * K::MPB + ml;                // mode within the i_z plane: iy (N/2 + 1) + ix
  const int iz = (int)blockIdx.y;
  const bool live = ml < (unsigned)K::MPB && q < plane;
  double2 acc[R];
#pragma unroll
  for (int r = 0; r < R; ++r) acc[r] = double2{0.0, 0.0};
  size_t m = 0;
  if (live) {
    const unsigned iy = q / nxh;
    const int ax = (int)(q - iy * nxh), ay = min((int)iy, N - (int)iy), az = min(iz, N - iz);
    m = (size_t)iz * plane + q;
    const double2* mrow = reinterpret_cast<const double2*>(M) + ((size_t)lin_class_of(ax, ay, az) * C + rp * R) * NF;
    double2 mm[R][NF];                                         // rows rp R .. rp R + R - 1 of M: R x 2 NF doubles, contiguous
#pragma unroll
    for (int r = 0; r < R; ++r) lin_load_row<NF>(mrow + r * NF, mm[r]);
#pragma unroll
    for (int c2 = 0; c2 < NF; ++c2) {
      const double2 u = __ldcs(dPhi + (size_t)c2 * nmodes + m);   // the modes stream through once: evict-first, the
      const double2 w = __ldcs(dPi + (size_t)c2 * nmodes + m);    // matrix table (47 MB at 256^3) stays in L2
#pragma unroll
      for (int r = 0; r < R; ++r) {
        acc[r].x = fma(mm[r][c2].x, u.x, acc[r].x); acc[r].y = fma(mm[r][c2].x, u.y, acc[r].y);
        acc[r].x = fma(mm[r][c2].y, w.x, acc[r].x); acc[r].y = fma(mm[r][c2].y, w.y, acc[r].y);
      }
    }
  }
  __syncthreads();                                             // every read of the block before its first write
  if (live) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const unsigned row = rp * R + r;
      __stcs(((row & 1) ? dPi : dPhi) + (size_t)(row >> 1) * nmodes + m, acc[r]);
    }
  }
}

// Every mode through every stage on its own ("naive version").  Real coefficients: the real and
// imaginary parts are two independent copies of the same system.
template <int NF>
__global__ void __launch_bounds__(kLinThreads)
lin_naive(double2* __restrict__ dPhi, double2* __restrict__ dPi, const LinStage<NF>* __restrict__ table, size_t nst,
          LinStencil sc, int N, size_t nmodes) {
  constexpr int W = 2 + NF * NF;
  __shared__ double sh[kLinChunk * W];
  size_t m;
  int ax, ay, az;
  const bool live = lin_mode_of_thread(N, m, ax, ay, az);
  double k2 = 0.0;
  double pr[NF], qr[NF], pim[NF], qim[NF];
#pragma unroll
  for (int i = 0; i < NF; ++i) pr[i] = qr[i] = pim[i] = qim[i] = 0.0;
  if (live) {
    k2 = lin_k_eff2(sc.c, N, ax, ay, az);
#pragma unroll
    for (int i = 0; i < NF; ++i) {
      const double2 a = dPhi[(size_t)i * nmodes + m], b = dPi[(size_t)i * nmodes + m];
      pr[i] = a.x; pim[i] = a.y; qr[i] = b.x; qim[i] = b.y;
    }
  }
  for (size_t base = 0; base < nst; base += kLinChunk) {
    const int n = (int)min((size_t)kLinChunk, nst - base);
    __syncthreads();
    lin_stage_chunk<NF>(table, base, n, sh);
    __syncthreads();
    if (live)
      for (int s = 0; s < n; ++s) {
        lin_stage<NF>(sh + s * W, k2, pr, qr);
        lin_stage<NF>(sh + s * W, k2, pim, qim);
      }
  }
  if (live) {
#pragma unroll
    for (int i = 0; i < NF; ++i) {
      dPhi[(size_t)i * nmodes + m] = double2{pr[i], pim[i]};
      dPi[(size_t)i * nmodes + m] = double2{qr[i], qim[i]};
    }
  }
}

// (2.22), reading G27: the k = 0 mode of every array is zero.
__global__ void lin_zero_mode(double2* dPhi, double2* dPi, int nf, size_t nmodes) {
  const int f = threadIdx.x;
  if (f < nf) { dPhi[(size_t)f * nmodes] = double2{0.0, 0.0}; dPi[(size_t)f * nmodes] = double2{0.0, 0.0}; }
}
__global__ void lin_scale(double* x, size_t n, double s) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) x[i] *= s;
}

}  // namespace pycool
