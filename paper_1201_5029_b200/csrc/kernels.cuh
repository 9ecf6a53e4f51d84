// kernels.cuh -- sm_100a kernels of the symplectic lattice step (arXiv 1201.5029 §2.3, eq. (2.47)-(2.48)).
//
//   kick_fused      one pass per stage: merged drift (H2 halves of two adjacent stages) + kick (H3) + the three
//                   lattice sums, 2.5D z-march with an x-y tile (+1 halo) in shared memory; register-prefetch
//                   loads, any N (the TMA-fed kernel for even N is kick_tma.cuh).
//   stage_finish    tail of either kick: the last block to finish adds the per-item partial sums in index order
//                   and advances (a, p_a) through H3, H2, H1 and the next stage's coefficients (scalar_advance)
//                   on the device (the paper does these on the CPU after a D2H copy).
//   scalar_update   the same as a stand-alone launch: opens a pycool_step call (and follows every kick when the
//                   fused tail is switched off).
//   drift_flush     deferred closing half drift phi += c pi, applied when phi is looked at.
//   sumsq / energy  lattice sums for set_fields and pycool_energies ((2.8), (2.16)).
//
// Layout [field][z][y][x], x fastest.  See DESIGN.md for the derivation of the merged drift, the register
// queue along z and the byte counts.
#pragma once
#include <cstddef>
#include <cstdint>

#include "potentials.cuh"

namespace pycool {

// ------------------------------------------------------------------------------------------------ layout
// Field arrays in HBM: [field][z][y + gy][x + gx], x fastest, rows `pitch` elements apart, `rows` rows per
// plane.  gx = gy = 0 is the plain N^3 layout.  With ghosts (gx = 16 bytes of elements, gy = 1) column x = -1
// holds the periodic image of x = N-1, x = N that of x = 0, likewise rows y = -1 and y = N, so that a TMA box
// with a one-site halo never leaves the array (kick_tma.cuh).  Every kernel that writes phi or pi keeps the
// images equal to their sources.
struct Layout {
  int N;
  int pitch, rows;
  int gx, gy;
  size_t plane;    // pitch * rows
  size_t field;    // plane * N
  size_t total;    // field * nf  (elements per array, padding included)
  __host__ __device__ __forceinline__ size_t at(int f, int z, int y, int x) const {
    return (size_t)f * field + (size_t)z * plane + (size_t)(y + gy) * pitch + (size_t)(x + gx);
  }
};

// Store v at site (x, y) of the (field, z) plane starting at `plane_base`, and at its periodic images in the
// ghost columns / rows.
template <typename Real>
__device__ __forceinline__ void store_site(Real* plane_base, const Layout& L, int x, int y, Real v) {
  Real* p = plane_base + (size_t)(y + L.gy) * L.pitch + (x + L.gx);
  *p = v;
  if (L.gx == 0) return;
  const bool xl = x < L.gx, xh = x >= L.N - L.gx, yl = y < L.gy, yh = y >= L.N - L.gy;
  if (!(xl | xh | yl | yh)) return;
  const long long dy = (long long)L.N * L.pitch;
  if (xl) p[L.N] = v;
  if (xh) p[-L.N] = v;
  if (yl) {
    p[dy] = v;
    if (xl) p[dy + L.N] = v;
    if (xh) p[dy - L.N] = v;
  }
  if (yh) {
    p[-dy] = v;
    if (xl) p[-dy + L.N] = v;
    if (xh) p[-dy - L.N] = v;
  }
}

// ------------------------------------------------------------------------------------------------ scalars
struct Scalars {          // device-resident; one per context
  double a, p_a;
  double Spi2, SD, SV;    // sum pi^2 (current pi), sum_f phi_f D[phi_f], sum V of the latest kick
  double c_drift;         // pending drift coefficient: phi += c_drift * pi before the next kick
  double kD, kV;          // a^2 h/dx^2 and a^4 h of the next kick
  double dt_cur;          // conformal length of the current step (= dt, or dt / a at its start when adaptive)
  double eta;             // conformal time: sum of the completed steps' lengths
  int nonfinite;          // sticky: a lattice sum was NaN/Inf
  int pad;
  // the time-synchronised state at the end of the latest completed step (a and p_a above already carry the opening
  // half flows of the next stage while a pycool_step call is under way): what an energy read-out at that instant
  // sees, and the closing half drift phi += c_close pi that makes phi synchronous with it (the energy log)
  double a_sync, pa_sync, c_close;
};

struct ScalarConst {
  double den;      // 6 V_L mpl^2  ((2.47) H1); +INF for a static background
  double Vrho_m;   // V_L rho_m0   ((2.47) H2)
  double dx2;      // dx^2
};

// Each operation below is a separate IEEE operation in the order the paper's flows (2.47) are written
// (no FMA contraction), so a and p_a differ from a plain evaluation only through the lattice sums.
__device__ __forceinline__ void flow_H1(Scalars& s, const ScalarConst& k, double e) {
  s.a = __dsub_rn(s.a, __dmul_rn(__ddiv_rn(s.p_a, k.den), e));                       // a -= p_a/(6 V mpl^2) e
}
__device__ __forceinline__ void flow_H2_pa(Scalars& s, const ScalarConst& k, double e) {
  const double a3 = __dmul_rn(__dmul_rn(s.a, s.a), s.a);
  s.p_a = __dadd_rn(s.p_a, __dmul_rn(__dsub_rn(__ddiv_rn(s.Spi2, a3), k.Vrho_m), e));   // (sum pi^2/a^3 - V rho_m) e
}
__device__ __forceinline__ double drift_coef(const Scalars& s, double e) {
  return __ddiv_rn(e, __dmul_rn(s.a, s.a));                                          // e / a^2
}
__device__ __forceinline__ void flow_H3_pa(Scalars& s, const ScalarConst& k, double e) {
  const double t1 = __ddiv_rn(__dmul_rn(s.a, s.SD), k.dx2);                          // a sum phi D phi / dx^2
  const double t2 = __dmul_rn(__dmul_rn(__dmul_rn(__dmul_rn(4.0, s.a), s.a), s.a), s.SV);   // 4 a^3 sum V
  s.p_a = __dadd_rn(s.p_a, __dmul_rn(__dsub_rn(t1, t2), e));
}
__device__ __forceinline__ void kick_coefs(Scalars& s, const ScalarConst& k, double h) {
  const double a2 = __dmul_rn(s.a, s.a);
  s.kD = __dmul_rn(__ddiv_rn(a2, k.dx2), h);
  s.kV = __dmul_rn(__dmul_rn(__dmul_rn(a2, s.a), s.a), h);
}

constexpr int kReduceThreads = 1024;

// Fixed-order sum of v[0..n) by one block of T threads: thread t adds elements t, t+T, t+2T, ... in order, then
// a shared-memory tree whose shape depends only on T.  Result valid in every thread.  Loads bypass L1 (the
// fused tail reads partial sums other blocks wrote during the same launch).
template <int T>
__device__ __forceinline__ double block_sum_fixed(const double* v, int n, double* sh /* T doubles */) {
  static_assert((T & (T - 1)) == 0, "tree shape: power of two");
  double acc = 0.0;
  for (int i = threadIdx.x; i < n; i += T) acc += __ldcg(v + i);
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = T / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
    __syncthreads();
  }
  const double r = sh[0];
  __syncthreads();
  return r;
}

// The three sums of a stage in one pass: the same per-quantity arithmetic as three block_sum_fixed calls (same strided
// partial sums, same tree), but one set of loads in flight and one barrier per tree level instead of three.
template <int T>
__device__ __forceinline__ void block_sum_fixed3(const double* v, size_t stride, int n, double* sh /* 3 T doubles */,
                                                 double (&out)[3]) {
  static_assert((T & (T - 1)) == 0 && T >= 64, "tree shape: power of two, at least two warps");
  double a0 = 0.0, a1 = 0.0, a2 = 0.0;
  for (int i = threadIdx.x; i < n; i += T) {
    a0 += __ldcg(v + i); a1 += __ldcg(v + stride + i); a2 += __ldcg(v + 2 * stride + i);
  }
  sh[threadIdx.x] = a0; sh[T + threadIdx.x] = a1; sh[2 * T + threadIdx.x] = a2;
  __syncthreads();
  for (int s = T / 2; s >= 32; s >>= 1) {                      // levels that cross warps: through shared memory
    if ((int)threadIdx.x < s) {
      sh[threadIdx.x] += sh[threadIdx.x + s];
      sh[T + threadIdx.x] += sh[T + threadIdx.x + s];
      sh[2 * T + threadIdx.x] += sh[2 * T + threadIdx.x + s];
    }
    __syncthreads();
  }
  if (threadIdx.x < 32) {                                      // the last five levels inside warp 0: lane i adds lane
    a0 = sh[threadIdx.x]; a1 = sh[T + threadIdx.x]; a2 = sh[2 * T + threadIdx.x];   // i + s, the tree's own pairs
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
      a0 += __shfl_down_sync(0xffffffffu, a0, s);
      a1 += __shfl_down_sync(0xffffffffu, a1, s);
      a2 += __shfl_down_sync(0xffffffffu, a2, s);
    }
    if (threadIdx.x == 0) { sh[0] = a0; sh[T] = a1; sh[2 * T] = a2; }
  }
  __syncthreads();
  out[0] = sh[0]; out[1] = sh[T]; out[2] = sh[2 * T];
  __syncthreads();
}

// Lengths of a stage and of the one after it, as weights of the step length.
struct StageLen {
  double w, w_next;   // stage weights (2.42)-(2.45), Table 1; w_next = 0: the call ends after this stage
  double dt;          // the fixed conformal step, or the physical-time increment when adaptive
  int adaptive;       // step length = dt / a(start of the step): "adaptive conformal step with constant
                      // increases in physical time"
  int ends_step;      // this stage is the last of its step
};

// Stage lengths of a multi-stage cooperative launch (kick_tma.cuh: kick_tma_coop): the device forms each StageLen.
struct CoopSchedule {
  double w[16];          // stage weights of one step (2.42)-(2.45), Table 1
  int ns;                // stages per step
  int first;             // index of this launch's first stage within the pycool_step call
  int nstages;           // stages in this launch
  int call_ends;         // the call ends with this launch: no stage follows the last one
  double dt;
  int adaptive;
};

// The scalar side of the step, one thread.
// mode 0: opening of a pycool_step call: H1(h_next/2), H2(h_next/2) scalar part, coefficients of the first kick.
// mode 2: the same, continuing from a call whose closing half drift h/(2 a^2) has not been applied yet
//         (s.c_drift): it merges with the opening half drift exactly as between two stages of one call.
// mode 1: after the kick of a stage of length h, given its reduced sums (SD, SV, Spi2): H3 p_a; H2(h/2) p_a;
//         H1(h/2); and, if h_next != 0, the opening of the next stage merged in: H1(h_next/2), H2(h_next/2) p_a,
//         c_drift = h/(2 a_i^2) + h_next/(2 a_{i+1}^2).
__device__ __forceinline__ void scalar_advance(Scalars& s, const ScalarConst& k, const StageLen& len, int mode,
                                               double SD, double SV, double SP) {
  const double step_len = len.adaptive ? s.dt_cur : len.dt;
  double c1 = mode == 2 ? s.c_drift : 0.0;     // mode 2: the previous call's closing half drift is still pending
  if (mode == 1) {
    const double h = __dmul_rn(len.w, step_len);
    s.SD = SD; s.SV = SV; s.Spi2 = SP;
    if (!(isfinite(SD) && isfinite(SV) && isfinite(SP))) s.nonfinite = 1;
    flow_H3_pa(s, k, h);                       // H3(h), scalar part
    const double e = __dmul_rn(h, 0.5);          // = h / 2 exactly (a power of two, h far from the subnormals): no division
    flow_H2_pa(s, k, e);                       // H2(h/2), scalar part (pi is constant in H2: post-kick sum)
    c1 = drift_coef(s, e);                     //          field part, applied by the next kernel
    flow_H1(s, k, e);                          // H1(h/2)
    if (len.ends_step) {
      s.eta = __dadd_rn(s.eta, step_len);
      s.a_sync = s.a; s.pa_sync = s.p_a; s.c_close = c1;
    }
  }
  if (len.w_next != 0.0) {
    double next_len = step_len;
    if (mode != 1 || len.ends_step) {          // a new step begins: its length from the a it starts with
      next_len = len.adaptive ? __ddiv_rn(len.dt, s.a) : len.dt;
      s.dt_cur = next_len;
    }
    const double h_next = __dmul_rn(len.w_next, next_len);
    const double e = __dmul_rn(h_next, 0.5);
    flow_H1(s, k, e);                          // H1(h_next/2)
    flow_H2_pa(s, k, e);                       // H2(h_next/2), scalar part
    s.c_drift = __dadd_rn(c1, drift_coef(s, e));
    kick_coefs(s, k, h_next);
  } else {
    s.c_drift = c1;
  }
}

// Tail of a kick kernel.  Thread 0 of every block publishes the block's three partial sums (index = linear
// block id, so the final order does not depend on arrival).  With a ticket counter (fused mode) the block that
// arrives last -- every other block has published by then -- reduces all partials in index order and advances
// the scalars: the stage needs no second launch.  The kernel's own reads of *sc all precede its ticket.
struct StageTail {
  Scalars* sc;
  unsigned int* ticket;   // blocks-done counter, zero between launches
  unsigned int* work;     // work-item claim counter of a persistent launch (kick_tma), zero between launches
  int fused;              // 0: partials only (scalar_update follows as its own launch)
  ScalarConst k;
  StageLen len;
};

// Thread 0: the three partial sums of work item `idx` of `nparts` (the order of the final sum is the index
// order, whichever block computed the item and whenever).
__device__ __forceinline__ void publish_partials(double* partials, unsigned nparts, unsigned idx,
                                                 const double (&v)[3]) {
  partials[idx] = v[0];
  partials[(size_t)nparts + idx] = v[1];
  partials[2 * (size_t)nparts + idx] = v[2];
}

// All threads, once per block, after thread 0 published the block's last partials.
template <int NT>
__device__ __forceinline__ void stage_finish(const StageTail& t, const double* partials, unsigned nparts,
                                             double* sh /* >= 3 NT doubles, free to overwrite */) {
  __shared__ int is_last;
  if (threadIdx.x == 0) {
    __threadfence();
    is_last = atomicAdd(t.ticket, 1u) == gridDim.x * gridDim.y * gridDim.z - 1;
  }
  __syncthreads();
  if (!is_last) return;
  if (threadIdx.x == 0) {                      // every block is done: counters ready for the next launch
    *t.ticket = 0u;
    *t.work = 0u;
  }
  if (!t.fused) return;
  __threadfence();
  double S3[3];
  block_sum_fixed3<NT>(partials, (size_t)nparts, (int)nparts, sh, S3);
  if (threadIdx.x == 0) {
    Scalars s = *t.sc;
    scalar_advance(s, t.k, t.len, 1, S3[0], S3[1], S3[2]);
    *t.sc = s;
  }
}

// One work item per block (kick_fused): publish, then finish.
template <int NT>
__device__ __forceinline__ void stage_tail(const StageTail& t, double* partials, const double (&v)[3], double* sh) {
  const unsigned nb = gridDim.x * gridDim.y * gridDim.z;
  const unsigned b = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
  if (threadIdx.x == 0) publish_partials(partials, nb, b, v);
  stage_finish<NT>(t, partials, nb, sh);
}

// ------------------------------------------------------------------------------------------------ block reduce
// Deterministic block reduction of NQ doubles per thread: warp shuffles (fixed pattern), then warp 0 lane 0
// adds the per-warp values in warp order.  Result valid in thread 0.
template <int NQ, int NT>
__device__ __forceinline__ void block_reduce(double (&v)[NQ], double* sh /* NQ * NT/32 */) {
  constexpr int NW = NT / 32;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_down_sync(0xffffffffu, v[q], o);
    if (lane == 0) sh[q * NW + warp] = v[q];
  }
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      double t = sh[q * NW];
      for (int w = 1; w < NW; ++w) t += sh[q * NW + w];
      v[q] = t;
    }
  }
}

// ------------------------------------------------------------------------------------------------ fused kick
template <typename Real>
struct KickArgs {
  const Real* phi_in;
  const Real* pi_in;
  Real* phi_out;
  Real* pi_out;
  const Scalars* sc;
  double* partials;      // [3][nblocks]: SD, SV, Spi2
  StageTail tail;        // fused reduction + scalar update by the last block
  Layout L;
  int zc;                // planes per z-chunk
  double c1, c2, c3;     // stencil weights by neighbour class (c0 = -(6c1+12c2+8c3))
  ModelParams mp;
};

template <int TX, int TY, int K>
struct Tile {
  static constexpr int kTX = TX, kTY = TY, kK = K;
  static constexpr int NT = TX * (TY / K);
  static constexpr int PX = TX + 2;                    // smem pitch
  static constexpr int PLANE = (TY + 2) * PX;          // smem elements per field per buffer
  static_assert(TY % K == 0, "K must divide TY");
  static_assert(2 * (TX + 2) + 2 * TY <= NT, "one halo site per thread at most");
  static_assert(NT % 32 == 0 && NT <= 1024, "block size");
};

template <typename Real, class Model, class T>
constexpr size_t kick_smem_bytes() {
  size_t tile = 2 * (size_t)Model::NF * T::PLANE * sizeof(Real);
  size_t red = 3 * (size_t)T::NT * sizeof(double);      // block_reduce scratch, then the tail's three trees
  return tile > red ? tile : red;
}

// One stage.  Block (bx,by,bz) owns outputs x in [bx TX, +TX), y in [by TY, +TY), z in [bz zc, +zc) (clipped
// to N) and marches z over planes z0-1 .. z0+nz.  For every plane it
//   1. drifts: phi' = phi + c_drift pi for the tile and its 1-site periodic halo (the merged H2 halves),
//      stores phi' (own planes only) and psi = phi' - ref_f into shared memory, ref_f a block-uniform value
//      of field f -- D annihilates constants, so D[psi] = D[phi'] but without cancellation against the
//      homogeneous part of the field;
//   2. forms the in-plane sums P0 (centre), P1 (4 faces), P2 (4 corners) of the plane, from which the
//      27-point stencil of three consecutive output planes is assembled in two running accumulators (A, B);
//   3. finalises output plane p-1: D, dV/dphi, pi' = pi + kD D - kV dV, the three sums.
// Thread (tx,ty) owns column x = tx and rows y = ty K .. ty K + K-1 of the tile.
template <typename Real, class Model, class T>
__global__ void __launch_bounds__(T::NT)
kick_fused(const KickArgs<Real> g) {
  constexpr int NF = Model::NF, K = T::kK, TX = T::kTX, TY = T::kTY, NT = T::NT, PX = T::PX;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Real* sm = reinterpret_cast<Real*>(smem_raw);          // [2][NF][TY+2][PX]

  const Layout& L = g.L;
  const int N = L.N;
  const size_t V = L.field;
  const int tid = threadIdx.x;
  const int tx = tid % TX, ty = tid / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * g.zc;
  const int wx = min(TX, N - x0), wy = min(TY, N - y0), nz = min(g.zc, N - z0);

  const Real cd = Real(g.sc->c_drift), kD = Real(g.sc->kD), kV = Real(g.sc->kV);
  const Real c1 = Real(g.c1), c2 = Real(g.c2), c3 = Real(g.c3);
  const Real c0 = -(Real(6) * c1 + Real(12) * c2 + Real(8) * c3);
  const typename Model::template Coef<Real> coef(g.mp);

  Real ref[NF];
#pragma unroll
  for (int f = 0; f < NF; ++f) ref[f] = g.phi_in[L.at(f, z0, y0, x0)];

  // own sites
  const int gx = x0 + tx;
  bool valid[K];
  size_t own_off[K];                                       // (y*N + x) of the K own sites
#pragma unroll
  for (int j = 0; j < K; ++j) {
    const int ly = ty * K + j;
    valid[j] = (tx < wx) && (ly < wy);
    own_off[j] = (size_t)(y0 + ly + L.gy) * L.pitch + gx + L.gx;
  }
  // halo site of this thread (ring of the (wy+2) x (wx+2) smem tile)
  const int nh = 2 * (wx + 2) + 2 * wy;
  const bool has_halo = tid < nh;
  int hsx = 0, hsy = 0;
  if (has_halo) {
    if (tid < wx + 2) { hsy = 0; hsx = tid; }
    else if (tid < 2 * (wx + 2)) { hsy = wy + 1; hsx = tid - (wx + 2); }
    else { const int r = tid - 2 * (wx + 2); hsy = 1 + (r >> 1); hsx = (r & 1) ? wx + 1 : 0; }
  }
  size_t halo_off;
  {
    int hx = x0 - 1 + hsx, hy = y0 - 1 + hsy;              // periodic wrap
    hx = hx < 0 ? hx + N : (hx >= N ? hx - N : hx);
    hy = hy < 0 ? hy + N : (hy >= N ? hy - N : hy);
    halo_off = (size_t)(hy + L.gy) * L.pitch + hx + L.gx;
  }

  Real rphi[NF][K], rpi[NF][K], hphi[NF], hpi[NF];         // loads in flight (plane p+1)
  Real pphi[NF][K], ppi[NF][K];                            // phi', pi of plane p-1 (to be finalised)
  Real cphi[NF][K], cpi[NF][K];                            // phi', pi of plane p
  Real A[NF][K], B[NF][K];                                 // stencil accumulators, see step 2
  double sD = 0.0, sV = 0.0, sP = 0.0;
#pragma unroll
  for (int f = 0; f < NF; ++f)
#pragma unroll
    for (int j = 0; j < K; ++j) { A[f][j] = B[f][j] = pphi[f][j] = ppi[f][j] = Real(0); }

  auto zplane = [&](int p) -> size_t {
    int gz = z0 + p;
    gz = gz < 0 ? gz + N : (gz >= N ? gz - N : gz);
    return (size_t)gz * L.plane;
  };
  auto load = [&](int p) {
    const size_t zp = zplane(p);
#pragma unroll
    for (int f = 0; f < NF; ++f) {
#pragma unroll
      for (int j = 0; j < K; ++j) {
        rphi[f][j] = Real(0); rpi[f][j] = Real(0);
        if (valid[j]) {
          const size_t i = f * V + zp + own_off[j];
          rphi[f][j] = __ldg(g.phi_in + i);
          rpi[f][j] = __ldg(g.pi_in + i);
        }
      }
      hphi[f] = Real(0); hpi[f] = Real(0);
      if (has_halo) {
        const size_t i = f * V + zp + halo_off;
        hphi[f] = __ldg(g.phi_in + i);
        hpi[f] = __ldg(g.pi_in + i);
      }
    }
  };

  load(-1);
#pragma unroll 1
  for (int p = -1; p <= nz; ++p) {
    Real* buf = sm + (size_t)((p + 1) & 1) * NF * T::PLANE;
    // ---- 1. drift + stage into shared memory
    const bool own_plane = (p >= 0) && (p < nz);
    const size_t zp = zplane(p);
#pragma unroll
    for (int f = 0; f < NF; ++f) {
#pragma unroll
      for (int j = 0; j < K; ++j) {
        const Real ph = fma(cd, rpi[f][j], rphi[f][j]);     // phi' = phi + c_drift pi
        cphi[f][j] = ph; cpi[f][j] = rpi[f][j];
        if (valid[j]) {
          if (own_plane) store_site(g.phi_out + f * V + zp, L, gx, y0 + ty * K + j, ph);
          buf[f * T::PLANE + (ty * K + j + 1) * PX + tx + 1] = ph - ref[f];
        }
      }
      if (has_halo) buf[f * T::PLANE + hsy * PX + hsx] = fma(cd, hpi[f], hphi[f]) - ref[f];
    }
    if (p < nz) load(p + 1);                                // in flight during the compute phase
    __syncthreads();

    // ---- 2. in-plane sums of plane p and 3. finalise plane p-1
    Real D[NF][K];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const Real* s = buf + f * T::PLANE + (ty * K) * PX + tx;
      Real R[K + 2], C[K + 2];
#pragma unroll
      for (int r = 0; r < K + 2; ++r) {
        const Real l = s[r * PX], c = s[r * PX + 1], rr = s[r * PX + 2];
        R[r] = l + rr; C[r] = c;
      }
#pragma unroll
      for (int j = 0; j < K; ++j) {
        const Real P0 = C[j + 1];
        const Real P1 = R[j + 1] + (C[j] + C[j + 2]);
        const Real P2 = R[j] + R[j + 2];
        const Real up = c1 * P0 + c2 * P1 + c3 * P2;        // weight of plane p in outputs p-1 and p+1
        const Real mid = c0 * P0 + c1 * P1 + c2 * P2;       // weight of plane p in output p
        D[f][j] = A[f][j] + up;                             // output p-1 complete
        A[f][j] = B[f][j] + mid;
        B[f][j] = up;
      }
    }
    if (p >= 1) {
      const size_t zq = zplane(p - 1);
#pragma unroll
      for (int j = 0; j < K; ++j) {
        if (valid[j]) {
          Real ph[NF], dV[NF];
#pragma unroll
          for (int f = 0; f < NF; ++f) ph[f] = pphi[f][j];
          const Real v = Model::template eval<Real>(coef, ph, dV);
          sV += (double)v;
#pragma unroll
          for (int f = 0; f < NF; ++f) {
            const Real pn = fma(kD, D[f][j], fma(-kV, dV[f], ppi[f][j]));   // pi' = pi + kD D - kV dV
            store_site(g.pi_out + f * V + zq, L, gx, y0 + ty * K + j, pn);
            sD = fma((double)ph[f], (double)D[f][j], sD);
            sP = fma((double)pn, (double)pn, sP);
          }
        }
      }
    }
#pragma unroll
    for (int f = 0; f < NF; ++f)
#pragma unroll
      for (int j = 0; j < K; ++j) { pphi[f][j] = cphi[f][j]; ppi[f][j] = cpi[f][j]; }
  }

  // ---- per-block partial sums, fixed order
  __syncthreads();
  double v[3] = {sD, sV, sP};
  block_reduce<3, NT>(v, reinterpret_cast<double*>(smem_raw));
  stage_tail<NT>(g.tail, g.partials, v, reinterpret_cast<double*>(smem_raw));
}

// ------------------------------------------------------------------------------------------------ pointwise
// Closing half drift of a pycool_step call: phi += c_drift pi, in place, over the whole padded array (ghost
// images of pi equal their sources, so the images of phi stay equal too).
template <typename Real>
__global__ void __launch_bounds__(256) drift_flush(Real* __restrict__ phi, const Real* __restrict__ pi,
                                                   const Scalars* __restrict__ sc, size_t n) {
  const Real cd = Real(sc->c_drift);
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
    phi[i] = fma(cd, pi[i], phi[i]);
}

// Periodic images into the ghost columns / rows of one array (after an upload).  One thread per padded site.
template <typename Real>
__global__ void __launch_bounds__(256) fill_ghosts(Real* __restrict__ v, Layout L, int nf) {
  const int W = L.N + 2 * L.gx, H = L.N + 2 * L.gy;
  const size_t per_plane = (size_t)W * H, n = per_plane * L.N * nf;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const size_t pl = i / per_plane;                       // f * N + z
    const int r = (int)(i - pl * per_plane);
    const int y = r / W - L.gy, x = r % W - L.gx;
    if (x >= 0 && x < L.N && y >= 0 && y < L.N) continue;
    int sx = x < 0 ? x + L.N : (x >= L.N ? x - L.N : x);
    int sy = y < 0 ? y + L.N : (y >= L.N ? y - L.N : y);
    sx = sx < 0 ? sx + L.N : (sx >= L.N ? sx - L.N : sx);  // N < gx (tiny lattices): wrap twice
    Real* base = v + pl * L.plane;
    base[(size_t)(y + L.gy) * L.pitch + (x + L.gx)] = base[(size_t)(sy + L.gy) * L.pitch + (sx + L.gx)];
  }
}

// sum of squares over the lattice sites (ghosts excluded) -> per-block partials (fixed assignment of elements
// to threads, fixed-order block reduce)
template <typename Real>
__global__ void __launch_bounds__(256) sumsq(const Real* __restrict__ v, Layout L, int nf,
                                             double* __restrict__ partials) {
  __shared__ double sh[8];
  double acc[1] = {0.0};
  const size_t n = (size_t)L.N * L.N * L.N * nf;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const size_t row = i / L.N;                            // (f * N + z) * N + y
    const int xx = (int)(i - row * L.N);
    const size_t pl = row / L.N;
    const int yy = (int)(row - pl * L.N);
    const double x = (double)v[pl * L.plane + (size_t)(yy + L.gy) * L.pitch + (xx + L.gx)];
    acc[0] = fma(x, x, acc[0]);
  }
  block_reduce<1, 256>(acc, sh);
  if (threadIdx.x == 0) partials[blockIdx.x] = acc[0];
}

// ------------------------------------------------------------------------------------------------ energies
// Per field: sum pi^2, sum G[phi] (2.8), sum phi D[phi] (2.7); and sum V.  One thread per site, direct
// (cached) neighbour loads; on-demand diagnostics, not the hot loop.
// partials: [3 NF + 1][gridDim.x]
template <typename Real, class Model>
__global__ void __launch_bounds__(256)
energy_sums(const Real* __restrict__ phi, const Real* __restrict__ pi, Layout L, double c1, double c2, double c3,
            ModelParams mp, double* __restrict__ partials, const Scalars* __restrict__ sc /* NULL: phi as stored */) {
  constexpr int NF = Model::NF, NQ = 3 * NF + 1;
  __shared__ double sh[NQ * 8];
  const int N = L.N;
  const size_t V = (size_t)N * N * N;
  const typename Model::template Coef<double> coef(mp);
  const double cw[4] = {0.0, c1, c2, c3};
  // with sc: the state seen through the pending closing half drift, phi' = phi + c_close pi, formed
  // in Real exactly as drift_flush would store it
  const bool drift = sc != nullptr;
  const Real cd = drift ? Real(sc->c_close) : Real(0);
  auto at = [&](const Real* pf, const Real* qf, size_t i) -> double {
    return drift ? (double)fma(cd, qf[i], pf[i]) : (double)pf[i];
  };
  double acc[NQ];
#pragma unroll
  for (int q = 0; q < NQ; ++q) acc[q] = 0.0;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += stride) {
    const int x = (int)(i % N), y = (int)((i / N) % N), z = (int)(i / ((size_t)N * N));
    int xs[3] = {x == 0 ? N - 1 : x - 1, x, x == N - 1 ? 0 : x + 1};
    int ys[3] = {y == 0 ? N - 1 : y - 1, y, y == N - 1 ? 0 : y + 1};
    int zs[3] = {z == 0 ? N - 1 : z - 1, z, z == N - 1 ? 0 : z + 1};
    double ph[NF], dV[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const Real* pf = phi + f * L.field;
      const Real* qf = pi + f * L.field;
      const size_t ic = L.at(0, z, y, x);
      const double ctr = at(pf, qf, ic);
      double s[4] = {0, 0, 0, 0}, q2[4] = {0, 0, 0, 0};
#pragma unroll
      for (int dz = 0; dz < 3; ++dz)
#pragma unroll
        for (int dy = 0; dy < 3; ++dy)
#pragma unroll
          for (int dx = 0; dx < 3; ++dx) {
            const int d = (dx != 1) + (dy != 1) + (dz != 1);
            if (d == 0) continue;
            const double df = at(pf, qf, L.at(0, zs[dz], ys[dy], xs[dx])) - ctr;
            s[d] += df;
            q2[d] = fma(df, df, q2[d]);
          }
      const double Dv = cw[1] * s[1] + cw[2] * s[2] + cw[3] * s[3];
      const double Gv = 0.5 * (cw[1] * q2[1] + cw[2] * q2[2] + cw[3] * q2[3]);
      const double pv = (double)pi[f * L.field + ic];
      acc[3 * f] = fma(pv, pv, acc[3 * f]);
      acc[3 * f + 1] += Gv;
      acc[3 * f + 2] = fma(ctr, Dv, acc[3 * f + 2]);
      ph[f] = ctr;
    }
    acc[3 * NF] += Model::template eval<double>(coef, ph, dV);
  }
  block_reduce<NQ, 256>(acc, sh);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) partials[(size_t)q * gridDim.x + blockIdx.x] = acc[q];
  }
}

}  // namespace pycool
