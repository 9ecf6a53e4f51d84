// kick_tma.cuh -- the fused drift + kick + lattice-sum stage of (2.47)-(2.48) as a TMA-fed z-march (sm_100a).
//
// Same arithmetic as kick_fused (kernels.cuh): per stage phi' = phi + c_drift pi, D = stencil (2.7) of phi',
// pi' = pi + kD D - kV dV/dphi(phi'), and the three sums of PAPER.md:327-331, 399.  What differs is how the
// planes reach the SM: one elected thread issues two 4-D tensor-map bulk copies (cp.async.bulk.tensor, SASS
// UTMALDG) per z-plane -- the (TX + 2G) x (TY + 2) x NF box of phi and of pi, halo included -- into a ring of
// S shared-memory stages that complete on mbarriers.  The loads in flight therefore live in shared memory, not
// in registers, and their depth (S - 1 planes ahead) is independent of occupancy.
//
// TMA boxes cannot wrap around a periodic lattice (out-of-bounds elements are zero-filled), so the arrays carry
// ghost images in x and y (Layout, kernels.cuh): every block writes, next to each output on a lattice face, its
// periodic image(s) into the ghost columns / rows of the output buffer, which the next stage then reads as plain
// in-bounds box elements.  z wraps through the box coordinate (one plane per box).  DESIGN.md "TMA path".
//
// Thread (txw, tyj) owns XW x J sites of the tile for all NF fields (default 2 x 2: x = 2 txw + {0,1}, y = 2 tyj + {0,1}).
#pragma once
#include <cuda.h>

#include <type_traits>

#include "kernels.cuh"

namespace pycool {

template <typename Real> struct Vec2T;
template <> struct Vec2T<double> { using type = double2; };
template <> struct Vec2T<float> { using type = float2; };

// XW consecutive sites along x, moved with one 8- or 16-byte access (float2, double2, float4).
template <typename Real, int XW>
struct alignas(XW * sizeof(Real) <= 16 ? XW * sizeof(Real) : 16) VecX {
  Real v[XW];
};

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
// 4-D tiled tensor-map load global -> shared, completion on an mbarrier (bytes of the whole box)
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2,
                                            int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::
          "r"(dst),
      "l"(reinterpret_cast<uint64_t>(tm)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

// Tile traits.  Thread (txw, tyj) owns the XW sites XW txw + {0 .. XW-1} of rows J tyj .. J tyj + J-1 for all
// fields (XW = 2: an x pair; XW = 4: an x quad, fp32 only -- one 16-byte access either way);
// MINB = blocks per SM the register budget is cut for (__launch_bounds__).
template <typename Real, int TX_, int TY_, int S_, int J_ = 2, int MINB_ = 1, int XW_ = 2>
struct TmaTile {
  static constexpr int TX = TX_, TY = TY_, S = S_, J = J_, MINB = MINB_, XW = XW_;
  static constexpr int G = 16 / (int)sizeof(Real);      // box halo / ghost columns on each side (16 bytes)
  static constexpr int PX = TX + 2 * G;                 // box row length
  static constexpr int RY = TY + 2;                     // box rows
  static constexpr int PLANE = PX * RY;                 // box elements per field
  static constexpr int NT = (TX / XW) * (TY / J);       // threads: XW x J sites each
  static constexpr int HR = (TX + 4) / 2;               // halo pairs in the top (and bottom) box row: x = -2 .. TX+1
  static constexpr int NHP = 2 * HR + 2 * TY;           // ring of halo pairs the stencil reads (x pairs)
  static_assert(TX % XW == 0 && TY % J == 0 && (J == 1 || J == 2 || J == 4), "XW x J sites per thread");
  static_assert(XW == 2 || (XW == 4 && sizeof(Real) == 4), "x quads: 16 bytes, so fp32 only");
  static_assert(NT % 32 == 0 && NT <= 1024, "block size");
  static_assert(PX <= 256 && RY <= 256, "TMA box extents");
};

// Box offsets of the halo pairs this thread converts every plane: the top and bottom box rows (x = -2 .. TX+1 in pairs)
// and the pairs left and right of every own row; -1 = none.  16-byte accesses in fp64, the outer element is unused.
template <class T>
__device__ __forceinline__ void halo_pairs_of_thread(int tid, int (&halo_sm)[(T::NHP + T::NT - 1) / T::NT]) {
  constexpr int NHT = (T::NHP + T::NT - 1) / T::NT;
#pragma unroll
  for (int k = 0; k < NHT; ++k) {
    const int h = tid + k * T::NT;
    int row, col;
    if (h < T::HR) { row = 0; col = T::G - 2 + 2 * h; }
    else if (h < 2 * T::HR) { row = T::TY + 1; col = T::G - 2 + 2 * (h - T::HR); }
    else { const int r = h - 2 * T::HR; row = 1 + (r >> 1); col = (r & 1) ? T::G + T::TX : T::G - 2; }
    halo_sm[k] = h < T::NHP ? row * T::PX + col : -1;
  }
}

template <typename Real, class Model, class T>
struct TmaSmem {
  static constexpr size_t BOX = (size_t)Model::NF * T::PLANE * sizeof(Real);   // bytes one bulk copy delivers
  static constexpr size_t BOXA = (BOX + 127) / 128 * 128;                      // 128-byte aligned slot
  static constexpr size_t RAW = (size_t)T::S * 2 * BOXA;                       // ring: [S][phi, pi]
  static constexpr size_t PSI = 2 * BOXA;                                      // double-buffered psi planes
  static constexpr size_t BARS = 128;                                          // S mbarriers
  static constexpr size_t RED = 3 * (T::NT / 32) * sizeof(double);             // per-item block reduction
  static constexpr size_t TOTAL = RAW + PSI + BARS + RED + 128;                // + slack to align the base
  static_assert(T::S * 8 <= BARS, "mbarriers fit");
  static_assert(3 * T::NT * sizeof(double) <= RAW + PSI, "the stage tail's three trees fit in the idle ring + psi");
  static constexpr bool kTreesFitPsi = 3 * T::NT * sizeof(double) <= PSI;   // kick_tma_coop: ring busy with the next stage
};

template <typename Real>
struct TmaArgs {
  Real* phi_out;
  Real* pi_out;
  const Scalars* sc;
  double* partials;       // [3][nitems]: SD, SV, Spi2
  StageTail tail;         // fused reduction + scalar update by the last block
  Layout L;
  int zc;                 // planes per z-chunk, at most (chunks are balanced: item_origin)
  int nbx, nby, nitems;   // work items = (x tile, y tile, z chunk): nitems = nbx nby nbz
  int ry;                 // item order: regions of ry rows of tiles, see item_origin (ry = nby: plain x-y-z order)
  double c1, c2, c3;
  ModelParams mp;
};

// Item index -> tile origin.  Items are numbered region by region -- a region is `ry` consecutive rows of x-y tiles
// (the last region may have fewer) -- and inside a region layer by layer in z, x fastest: all z-chunks of a region
// come before the next region.  The host sizes a region to about as many tiles as there are blocks in flight, so
// the blocks that finish layer k of a region claim layer k+1 of the same tiles next: chunk k+1 of a tile starts just
// when chunk k ends, the two planes they share as halo (top halo of k = first own plane of k+1, last own plane of k
// = bottom halo of k+1) are read twice within a few microseconds, and the second read hits L2.  In plain x-y-z
// order (ry = nby) the second read comes ~1.7 rounds (> 300 MB of traffic) later, always from DRAM: 12.5 % of the
// reads at 16-plane chunks (measured at 512^3: 4.88 -> 4.40 GB read per launch, 1.454 -> 1.405 ms, profiles/r2).
// Blocks in flight are still x-y neighbours within their layer (halo rows hit L2 as before).
// z-chunks are balanced: chunk bz of nbz owns planes [bz N / nbz, (bz + 1) N / nbz), lengths differing by one at most
// (128^3 on 148 SMs: 9 chunks of 14-15 planes x 16 tiles = 144 items in one round, instead of 8 x 16).
template <typename Real, int TX, int TY>
__device__ __forceinline__ void item_origin(const TmaArgs<Real>& g, int item, int& x0, int& y0, int& z0, int& nz) {
  const int nbz = g.nitems / (g.nbx * g.nby);
  const int per_region = g.ry * g.nbx * nbz;                   // every region but the last is full
  const int reg = item / per_region, r = item - reg * per_region;
  const int row0 = reg * g.ry;
  const int layer = min(g.ry, g.nby - row0) * g.nbx;           // tiles of one z-layer of this region
  const int bz = r / layer, t = r - bz * layer;
  const int ty = t / g.nbx, tx = t - ty * g.nbx;
  x0 = tx * TX; y0 = (row0 + ty) * TY;
  z0 = (int)(((long long)bz * g.L.N) / nbz);
  nz = (int)(((long long)(bz + 1) * g.L.N) / nbz) - z0;
}

// The z-march of one work item.  EDGE (compile time) = the item touches a lattice face or a ragged edge: only
// that copy carries the periodic-image stores and the validity predicates; interior items run branch-free.
template <bool EDGE, typename Real, class Model, class T, class IssueF>
__device__ __forceinline__ void march_item(const TmaArgs<Real>& g, Real* phi_out, Real* pi_out, IssueF& issue_next,
                                           int& slot, uint32_t& phase, unsigned char* raw, Real* psi,
                                           const uint32_t bars, const int x0,
                                           const int y0, const int z0, const int nz, const int own_sm,
                                           const int (&halo_sm)[(T::NHP + T::NT - 1) / T::NT], const Real cd,
                                           const Real kD, const Real kV, const Real c0, const Real c1, const Real c2,
                                           const Real c3, const typename Model::template Coef<Real>& coef,
                                           double& sD, double& sV, double& sP) {
  using R2 = typename Vec2T<Real>::type;                     // halo ring: always x pairs
  constexpr int XW = T::XW;
  using RV = VecX<Real, XW>;                                 // own sites: XW along x, one access
  using SM = TmaSmem<Real, Model, T>;
  constexpr int NF = Model::NF, TX = T::TX, TY = T::TY, S = T::S, G = T::G, PX = T::PX, NT = T::NT, J = T::J;
  constexpr int PLANE = T::PLANE;
  constexpr uint32_t ES = (uint32_t)sizeof(Real);
  constexpr int NHT = (T::NHP + NT - 1) / NT;
  const Layout& L = g.L;
  const int N = L.N;
  const int tid = threadIdx.x;
  const int txw = tid % (TX / XW), tyj = tid / (TX / XW);
  const size_t plane_b = L.plane * ES, field_b = L.field * ES;
  (void)TY; (void)S; (void)tyj;

  // lattice planes of the outputs p (phi') and p-1 (pi'), carried along the march instead of being wrapped anew
  // from z0 + p every plane
  int gz_cur = z0 - 1 < 0 ? z0 - 1 + N : z0 - 1, gz_prev = gz_cur;   // plane p = -1

  // Own sites.  Items that touch no lattice face and no ragged edge (block-uniform test) store through a
  // uniform plane pointer plus a 32-bit per-thread byte offset and nothing else; the others also write the
  // periodic images of their face sites into the ghost columns / rows and predicate ragged sites.
  // (XW never exceeds the ghost width L.gx = 16 bytes of elements, so a group is all image or no image.)
  const int gx = x0 + XW * txw;
  const bool okx = gx < N;
  int ximg = 0;                                              // element offset of the x image, 0 = none
  if (gx < L.gx) ximg = N; else if (gx >= N - L.gx) ximg = -N;
  const bool ximg2 = (gx < L.gx) && (gx >= N - L.gx);        // both images (N <= 2 gx only)
  bool valid[J];
  uint32_t own_off[J];                                       // byte offset within a (field, z) plane
  long long yimg[J];                                         // element offset of the y image, 0 = none
#pragma unroll
  for (int j = 0; j < J; ++j) {
    const int gy = y0 + J * tyj + j;
    valid[j] = okx && gy < N;
    own_off[j] = ((uint32_t)(gy + L.gy) * (uint32_t)L.pitch + (uint32_t)(gx + L.gx)) * ES;
    yimg[j] = 0;
    if (gy == 0) yimg[j] = (long long)N * L.pitch; else if (gy == N - 1) yimg[j] = -(long long)N * L.pitch;
  }
  auto store_edge = [&](unsigned char* plane, int j, RV v) { // one output group and its periodic images
    Real* p = reinterpret_cast<Real*>(plane + own_off[j]);
    *reinterpret_cast<RV*>(p) = v;
    if (ximg) {
      *reinterpret_cast<RV*>(p + ximg) = v;
      if (ximg2) *reinterpret_cast<RV*>(p - ximg) = v;
    }
    if (yimg[j]) {
      *reinterpret_cast<RV*>(p + yimg[j]) = v;
      if (ximg) {
        *reinterpret_cast<RV*>(p + yimg[j] + ximg) = v;
        if (ximg2) *reinterpret_cast<RV*>(p + yimg[j] - ximg) = v;
      }
    }
  };
  auto store_own = [&](unsigned char* plane, int j, RV v) {  // plain store (st.global.cs measured 9 % slower)
    if constexpr (!EDGE) *reinterpret_cast<RV*>(plane + own_off[j]) = v;
    else if (valid[j]) store_edge(plane, j, v);
  };

  // The stencil's single-element loads of the x-neighbours (x = -1 and x = XW of the thread's group) run at the group
  // stride, XW elements: threads 128 / (XW sizeof(Real)) apart hit the same banks, a 2-way conflict that costs the load
  // as many shared-memory wavefronts as the full-width load of the group itself.  Every other such run of threads takes
  // the RIGHT neighbour first and the left one second: the two halves then fall on disjoint banks in both loads.
  constexpr int NB_RUN = 128 / (XW * (int)sizeof(Real));
  const bool nb_swap = ((txw / NB_RUN) & 1) != 0;
  const int nb_first = nb_swap ? XW : -1, nb_second = nb_swap ? -1 : XW;

  RV qa_phi[NF][J], qa_pi[NF][J], qb_phi[NF][J], qb_pi[NF][J];  // phi', pi of planes p and p-1 (roles swap)
  RV A[NF][J], B[NF][J];                                     // stencil accumulators
  Real ref[NF];                                              // item-uniform; D annihilates constants
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    ref[f] = Real(0);
#pragma unroll
    for (int j = 0; j < J; ++j)
#pragma unroll
      for (int k = 0; k < XW; ++k)
        A[f][j].v[k] = B[f][j].v[k] = qa_phi[f][j].v[k] = qa_pi[f][j].v[k] = qb_phi[f][j].v[k] = qb_pi[f][j].v[k] = Real(0);
  }

  // One plane of the march: cphi/cpi receive plane p, pphi/ppi hold plane p-1 (finalised here).
  // EDGE (compile-time) = the item touches a lattice face or a ragged edge; interior items run a copy of the
  // march without any of the image / validity branches.
  auto step = [&](const int p, const int par, RV (&cphi)[NF][J], RV (&cpi)[NF][J], const RV (&pphi)[NF][J],
                  const RV (&ppi)[NF][J]) {
    const int s = slot;
    const Real* rphi = reinterpret_cast<const Real*>(raw + (size_t)s * 2 * SM::BOXA);
    const Real* rpi = reinterpret_cast<const Real*>(raw + (size_t)s * 2 * SM::BOXA + SM::BOXA);
    Real* pb = psi + (size_t)par * (SM::BOXA / sizeof(Real));
    mbar_wait(bars + 8u * s, phase);
    if (++slot == S) { slot = 0; phase ^= 1u; }

    // reference value of each field: phi at the item's first site one plane below (any item-uniform value
    // near the field does; it is the same for every thread because it is read from the shared box)
    if (p == -1) {
#pragma unroll
      for (int f = 0; f < NF; ++f) ref[f] = rphi[f * PLANE + PX + G];
    }

    // ---- 1. drift: phi' = phi + c_drift pi (own groups and halo ring); psi = phi' - ref to shared memory
    const bool own_plane = (p >= 0) && (p < nz);
    unsigned char* ophi = reinterpret_cast<unsigned char*>(phi_out) + (size_t)gz_cur * plane_b;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
#pragma unroll
      for (int j = 0; j < J; ++j) {
        const int o = f * PLANE + own_sm + j * PX;
        const RV a = *reinterpret_cast<const RV*>(rphi + o);
        const RV b = *reinterpret_cast<const RV*>(rpi + o);
        RV ph, ps;
#pragma unroll
        for (int k = 0; k < XW; ++k) {
          ph.v[k] = fma(cd, b.v[k], a.v[k]);
          ps.v[k] = ph.v[k] - ref[f];
        }
        cphi[f][j] = ph; cpi[f][j] = b;
        if (own_plane) store_own(ophi + f * field_b, j, ph);
        *reinterpret_cast<RV*>(pb + o) = ps;
      }
#pragma unroll
      for (int k = 0; k < NHT; ++k)
        if (halo_sm[k] >= 0) {
          const int o = f * PLANE + halo_sm[k];
          const R2 a = *reinterpret_cast<const R2*>(rphi + o);
          const R2 b = *reinterpret_cast<const R2*>(rpi + o);
          *reinterpret_cast<R2*>(pb + o) = R2{fma(cd, b.x, a.x) - ref[f], fma(cd, b.y, a.y) - ref[f]};
        }
    }
    __syncthreads();                                         // psi plane complete; raw stage s consumed
    issue_next(s);

    // ---- 2. in-plane sums of plane p; 3. finalise plane p-1
    RV D[NF][J];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const Real* sp = pb + f * PLANE + own_sm - PX;         // row above the first own row
      Real Sd[J + 2][XW], Ce[J + 2][XW];                     // per row and x-output: side sum (left + right), centre
#pragma unroll
      for (int r = 0; r < J + 2; ++r) {
        Real e[XW + 2];                                      // x = -1 .. XW of this row
        const Real n0 = sp[r * PX + nb_first], n1 = sp[r * PX + nb_second];   // the two neighbours, see nb_swap
        if (J >= 2 && r >= 1 && r <= J) {                    // an own row: its psi is phi' - ref of this thread's own
#pragma unroll                                               // registers, the very operation the drift stored -- no load
          for (int k = 0; k < XW; ++k) e[k + 1] = cphi[f][r - 1].v[k] - ref[f];   // (one-row variants: no gain measured,
        } else {                                             // and their 128-register budget is full)
          const RV m = *reinterpret_cast<const RV*>(sp + r * PX);
#pragma unroll
          for (int k = 0; k < XW; ++k) e[k + 1] = m.v[k];
        }
        e[0] = nb_swap ? n1 : n0;
        e[XW + 1] = nb_swap ? n0 : n1;
#pragma unroll
        for (int k = 0; k < XW; ++k) { Sd[r][k] = e[k] + e[k + 2]; Ce[r][k] = e[k + 1]; }
      }
#pragma unroll
      for (int j = 0; j < J; ++j) {
#pragma unroll
        for (int k = 0; k < XW; ++k) {
          const Real P0 = Ce[j + 1][k], P1 = Sd[j + 1][k] + (Ce[j][k] + Ce[j + 2][k]), P2 = Sd[j][k] + Sd[j + 2][k];
          const Real up = fma(c3, P2, fma(c2, P1, c1 * P0));  // weight of plane p in outputs p-1 and p+1
          D[f][j].v[k] = A[f][j].v[k] + up;                  // output p-1 complete
          A[f][j].v[k] = fma(c2, P2, fma(c1, P1, fma(c0, P0, B[f][j].v[k])));   // + weight of plane p in output p
          B[f][j].v[k] = up;
        }
      }
    }
    if (p >= 1) {
      unsigned char* opi = reinterpret_cast<unsigned char*>(pi_out) + (size_t)gz_prev * plane_b;   // plane p-1
#pragma unroll
      for (int j = 0; j < J; ++j) {
        if (!EDGE || valid[j]) {
          RV pn[NF];
#pragma unroll
          for (int k = 0; k < XW; ++k) {
            Real ph[NF], dV[NF];
#pragma unroll
            for (int f = 0; f < NF; ++f) ph[f] = pphi[f][j].v[k];
            sV += (double)Model::template eval<Real>(coef, ph, dV);
#pragma unroll
            for (int f = 0; f < NF; ++f) {
              pn[f].v[k] = fma(kD, D[f][j].v[k], fma(-kV, dV[f], ppi[f][j].v[k]));   // pi' = pi + kD D - kV dV
              sD = fma((double)ph[f], (double)D[f][j].v[k], sD);
              sP = fma((double)pn[f].v[k], (double)pn[f].v[k], sP);
            }
          }
#pragma unroll
          for (int f = 0; f < NF; ++f) store_own(opi + f * field_b, j, pn[f]);
        }
      }
    }
    gz_prev = gz_cur;                                        // on to plane p+1
    if (++gz_cur == N) gz_cur = 0;
  };

#pragma unroll 1
  for (int p = -1; p <= nz; p += 2) {                        // two planes per trip: the p / p-1 roles swap
    step(p, 0, qa_phi, qa_pi, qb_phi, qb_pi);
    if (p + 1 <= nz) step(p + 1, 1, qb_phi, qb_pi, qa_phi, qa_pi);
  }
}

// Work items.  With gridDim.x = nitems every block has one item.  With fewer blocks (as many as are resident on
// the GPU at once) the launch is persistent: a block's first item is its index, every further one is claimed
// from a device counter a few planes before the current item's loads run out -- the order in which a hardware
// block scheduler would hand them out, so the blocks in flight stay x-y neighbours within a few planes of each
// other (their halo rows hit L2), however unequal the SMs' speeds.  (A fixed round-robin deal loses that: blocks
// drift apart over ~28 items and DRAM reads grow 1.35x, measured.)  The TMA ring runs on across item
// boundaries: the first planes of the next item are in flight while the last planes of the current one are
// computed, so a block waits for a cold pipeline only once per launch.  Partial sums are indexed by item, so
// results do not depend on which block computed what.
template <typename Real, class Model, class T>
__global__ void __launch_bounds__(T::NT, T::MINB)
kick_tma(const __grid_constant__ CUtensorMap tm_phi, const __grid_constant__ CUtensorMap tm_pi,
         const TmaArgs<Real> g) {
  using SM = TmaSmem<Real, Model, T>;
  constexpr int TX = T::TX, TY = T::TY, S = T::S, G = T::G, PX = T::PX, NT = T::NT, J = T::J, XW = T::XW;

  extern __shared__ unsigned char smem_dyn[];
  unsigned char* base = smem_dyn + ((128u - (smem_addr(smem_dyn) & 127u)) & 127u);
  unsigned char* raw = base;                                   // [S][2][BOXA]
  Real* psi = reinterpret_cast<Real*>(base + SM::RAW);         // [2][BOXA]
  const uint32_t bars = smem_addr(base + SM::RAW + SM::PSI);   // S x 8 bytes
  double* red = reinterpret_cast<double*>(base + SM::RAW + SM::PSI + SM::BARS);

  const Layout& L = g.L;
  const int N = L.N;
  const int tid = threadIdx.x;
  const int txw = tid % (TX / XW), tyj = tid / (TX / XW);

  // ---- producer: the stream of loads, item after item, planes z0-1 .. z0+nz of each.  Every thread keeps the
  // (block-uniform) bookkeeping; only thread 0 touches the barriers, the TMA unit and the claim counter.
  __shared__ int item_ring[4];                                 // items of this block by sequence number (mod 4)
  const bool dyn = (int)gridDim.x < g.nitems;
  int pr_item = blockIdx.x, pr_seq = 0, pr_i = 0, pr_x0 = 0, pr_y0 = 0, pr_z0 = 0, pr_nload = 0;
  bool pr_switch = false;                                      // current item's loads all issued
  int claimed = 0x7fffffff;                                    // thread 0: the next item (none unless dyn)
  auto pr_decode = [&]() {
    if (pr_item < g.nitems) {
      int nz_;
      item_origin<Real, TX, TY>(g, pr_item, pr_x0, pr_y0, pr_z0, nz_);
      pr_nload = nz_ + 2;
    }
    pr_i = 0;
  };
  // Next load of the stream into ring slot s.  Call only after a block-wide barrier that follows the previous
  // call (the item switch reads what thread 0 wrote during that call).
  auto issue_next = [&](int s) {
    if (pr_switch) {
      pr_switch = false;
      pr_item = item_ring[++pr_seq & 3];
      pr_decode();
    }
    if (pr_item >= g.nitems) return;
    if (tid == 0) {
      const uint32_t bar = bars + 8u * s;
      const uint32_t dst = smem_addr(raw + (size_t)s * 2 * SM::BOXA);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(bar, (uint32_t)(2 * SM::BOX));
      int gz = pr_z0 + pr_i - 1;
      gz = gz < 0 ? gz + N : (gz >= N ? gz - N : gz);
      tma_load_4d(dst, &tm_phi, bar, pr_x0, pr_y0, gz, 0);     // box origin (x0-G, y0-1) in padded coordinates
      tma_load_4d(dst + (uint32_t)SM::BOXA, &tm_pi, bar, pr_x0, pr_y0, gz, 0);
      // claim the next item a few planes ahead, so the counter's round trip is over when the value is needed
      if (dyn && pr_i == max(pr_nload - 4, 0)) claimed = (int)(gridDim.x + atomicAdd(g.tail.work, 1u));
    }
    if (++pr_i == pr_nload) {
      if (tid == 0) item_ring[(pr_seq + 1) & 3] = claimed;     // INT_MAX ends the stream
      pr_switch = true;
    }
  };

  // Programmatic dependent launch: the next stage's grid may be scheduled while this one drains (its blocks take
  // the SMs this grid's blocks leave, set up their barriers and indices, then wait below), which hides the launch
  // latency and the prologue behind this grid's tail -- the last block's reduction and scalar update.  Nothing
  // above the wait reads what the previous stage wrote (fields, scalars, partials, counters).
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if (tid == 0) {
    for (int s = 0; s < S; ++s) mbar_init(bars + 8u * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  pr_decode();
  asm volatile("griddepcontrol.wait;" ::: "memory");           // previous kernel complete, its writes visible
  for (int s = 0; s < S; ++s) {
    issue_next(s);
    __syncthreads();                                           // also: barriers initialised before anyone waits
  }

  const Real cd = Real(g.sc->c_drift), kD = Real(g.sc->kD), kV = Real(g.sc->kV);
  const Real c1 = Real(g.c1), c2 = Real(g.c2), c3 = Real(g.c3);
  const Real c0 = -(Real(6) * c1 + Real(12) * c2 + Real(8) * c3);
  const typename Model::template Coef<Real> coef(g.mp);

  // box offsets: own pair of row j, and the halo pair(s) of this thread (top and bottom box rows x = -2 ..
  // TX+1, and the pairs left and right of every own row; 16-byte accesses, the outer element is unused)
  const int own_sm = (J * tyj + 1) * PX + G + XW * txw;
  constexpr int NHT = (T::NHP + NT - 1) / NT;                  // halo pairs per thread
  int halo_sm[NHT];
  halo_pairs_of_thread<T>(tid, halo_sm);
  int slot = 0;                                                // ring slot and phase of the next plane to consume
  uint32_t phase = 0;

  int cs_seq = 0;
#pragma unroll 1
  for (int item = blockIdx.x; item < g.nitems; item = item_ring[++cs_seq & 3]) {
    int x0, y0, z0, nz;
    item_origin<Real, TX, TY>(g, item, x0, y0, z0, nz);
    const bool edge_blk = (x0 < L.gx) | (x0 + TX > N - L.gx) | (y0 == 0) | (y0 + TY >= N);
    double sD = 0.0, sV = 0.0, sP = 0.0;
    if (edge_blk)
      march_item<true, Real, Model, T>(g, g.phi_out, g.pi_out, issue_next, slot, phase, raw, psi, bars, x0, y0, z0, nz,
                                       own_sm, halo_sm, cd, kD, kV, c0, c1, c2, c3, coef, sD, sV, sP);
    else
      march_item<false, Real, Model, T>(g, g.phi_out, g.pi_out, issue_next, slot, phase, raw, psi, bars, x0, y0, z0, nz,
                                        own_sm, halo_sm, cd, kD, kV, c0, c1, c2, c3, coef, sD, sV, sP);

    // ---- the item's partial sums, fixed order.  The barrier inside block_reduce also separates this item's
    // last reads of the psi planes from the next item's first writes.
    double v[3] = {sD, sV, sP};
    block_reduce<3, NT>(v, red);
    if (tid == 0) publish_partials(g.partials, (unsigned)g.nitems, (unsigned)item, v);
  }

  __syncthreads();                                             // ring (every load consumed) and psi are free: the tail's
  stage_finish<NT>(g.tail, g.partials, (unsigned)g.nitems, reinterpret_cast<double*>(raw));   // trees use them
}


// ------------------------------------------------------------------------------------------------ small lattices
// Several stages in ONE cooperative launch, for lattices whose work items all fit on the GPU at once (32^3 .. 128^3):
// one block per item, and between stages a grid-wide barrier instead of a kernel boundary -- the blocks stay
// resident, keep their shared-memory carve-up, barriers and per-thread tables, and a stage costs no launch
// hand-over (the paper returns to the CPU at every sub-step).  The barrier is the stage tail itself:
// every block publishes its partial sums and arrives on a counter in global memory; once all have, EVERY block adds
// the partials in item order and advances its own copy of the scalars (scalar_advance, as stage_finish does) -- the
// same operations on the same numbers everywhere, hence the same bits, and no second round trip through one "last"
// block -- while its first loads of the next stage are already in flight.  Same items, same partial-sum indices, same
// order of the final sum as the launch-per-stage path: results are bitwise identical (tested).  Needs
// cudaLaunchCooperativeKernel (co-residency).
template <typename Real>
struct CoopArgs {
  Real* phi[2];          // the two state buffers; stage k reads buffer (cur0 + k) & 1 and writes the other
  Real* pi[2];
  int cur0;
  unsigned int* release; // arrivals at the stage barriers of this launch, all blocks (zero at launch)
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_u32(unsigned* p, unsigned v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <typename Real, class Model, class T>
__global__ void __launch_bounds__(T::NT, T::MINB)
kick_tma_coop(const __grid_constant__ CUtensorMap tm_phi0, const __grid_constant__ CUtensorMap tm_pi0,
              const __grid_constant__ CUtensorMap tm_phi1, const __grid_constant__ CUtensorMap tm_pi1,
              const TmaArgs<Real> g, const CoopArgs<Real> ca, const CoopSchedule sch) {
  using SM = TmaSmem<Real, Model, T>;
  constexpr int TX = T::TX, TY = T::TY, S = T::S, G = T::G, PX = T::PX, NT = T::NT, J = T::J, XW = T::XW;

  extern __shared__ unsigned char smem_dyn[];
  unsigned char* base = smem_dyn + ((128u - (smem_addr(smem_dyn) & 127u)) & 127u);
  unsigned char* raw = base;
  Real* psi = reinterpret_cast<Real*>(base + SM::RAW);
  const uint32_t bars = smem_addr(base + SM::RAW + SM::PSI);
  double* red = reinterpret_cast<double*>(base + SM::RAW + SM::PSI + SM::BARS);
  static_assert(SM::kTreesFitPsi, "the stage tail's trees live in the psi planes while the ring refills");
  __shared__ Scalars sc_sh;                                    // this block's copy of the scalars (thread 0 advances it)
  __shared__ Real coef_sh[3];                                  // c_drift, kD, kV of the coming stage, in Real

  const Layout& L = g.L;
  const int N = L.N;
  const int tid = threadIdx.x;
  const int txw = tid % (TX / XW), tyj = tid / (TX / XW);
  const int item = blockIdx.x;                                 // one item per block, the same in every stage
  int x0, y0, z0, nz;
  item_origin<Real, TX, TY>(g, item, x0, y0, z0, nz);
  const bool edge_blk = (x0 < L.gx) | (x0 + TX > N - L.gx) | (y0 == 0) | (y0 + TY >= N);

  if (tid == 0) {
    for (int s = 0; s < S; ++s) mbar_init(bars + 8u * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    // the scalars the previous launch left: through L2 (this SM's L1 may hold an older copy)
    const double* src = reinterpret_cast<const double*>(g.sc);
    double* dst = reinterpret_cast<double*>(&sc_sh);
    static_assert(sizeof(Scalars) % sizeof(double) == 0, "Scalars is copied as doubles");
    for (int q = 0; q < (int)(sizeof(Scalars) / sizeof(double)); ++q) dst[q] = __ldcg(src + q);
    coef_sh[0] = Real(sc_sh.c_drift); coef_sh[1] = Real(sc_sh.kD); coef_sh[2] = Real(sc_sh.kV);
  }
  const Real c1 = Real(g.c1), c2 = Real(g.c2), c3 = Real(g.c3);
  const Real c0 = -(Real(6) * c1 + Real(12) * c2 + Real(8) * c3);
  const typename Model::template Coef<Real> coef(g.mp);
  const int own_sm = (J * tyj + 1) * PX + G + XW * txw;
  constexpr int NHT = (T::NHP + NT - 1) / NT;
  int halo_sm[NHT];
  halo_pairs_of_thread<T>(tid, halo_sm);
  int slot = 0;
  uint32_t phase = 0;
  __syncthreads();                                             // barriers initialised before anyone waits

  // the loads of a stage: planes z0-1 .. z0+nz of the block's item, S in flight
  const CUtensorMap* tphi = nullptr;
  const CUtensorMap* tpi = nullptr;
  int pr_i = 0;
  const int pr_nload = nz + 2;
  auto issue_next = [&](int s) {
    if (pr_i >= pr_nload) return;
    if (tid == 0) {
      const uint32_t bar = bars + 8u * s;
      const uint32_t dst = smem_addr(raw + (size_t)s * 2 * SM::BOXA);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(bar, (uint32_t)(2 * SM::BOX));
      int gz = z0 + pr_i - 1;
      gz = gz < 0 ? gz + N : (gz >= N ? gz - N : gz);
      tma_load_4d(dst, tphi, bar, x0, y0, gz, 0);
      tma_load_4d(dst + (uint32_t)SM::BOXA, tpi, bar, x0, y0, gz, 0);
    }
    ++pr_i;
  };
  // First loads of a stage (up to S, ring slots in consumption order from `slot`): thread 0 issues them -- one proxy
  // fence for all -- as soon as IT may (the ring is idle: every thread is past the march's last barrier), the others
  // only keep the books.
  auto start_loads = [&](int cur) {
    tphi = cur ? &tm_phi1 : &tm_phi0;
    tpi = cur ? &tm_pi1 : &tm_pi0;
    pr_i = pr_nload < S ? pr_nload : S;
  };
  auto issue_first = [&](int cur) {                            // thread 0 only
    const CUtensorMap* tp = cur ? &tm_phi1 : &tm_phi0;
    const CUtensorMap* tq = cur ? &tm_pi1 : &tm_pi0;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    const int n = pr_nload < S ? pr_nload : S;
    for (int i = 0; i < n; ++i) {
      int sl = slot + i; if (sl >= S) sl -= S;
      const uint32_t bar = bars + 8u * sl;
      const uint32_t dst = smem_addr(raw + (size_t)sl * 2 * SM::BOXA);
      mbar_expect_tx(bar, (uint32_t)(2 * SM::BOX));
      int gz = z0 + i - 1;
      gz = gz < 0 ? gz + N : (gz >= N ? gz - N : gz);
      tma_load_4d(dst, tp, bar, x0, y0, gz, 0);
      tma_load_4d(dst + (uint32_t)SM::BOXA, tq, bar, x0, y0, gz, 0);
    }
  };
  if (tid == 0) issue_first(ca.cur0 & 1);
  start_loads(ca.cur0 & 1);

#pragma unroll 1
  for (int k = 0; k < sch.nstages; ++k) {
    const int cur = (ca.cur0 + k) & 1;
    const Real cd = coef_sh[0], kD = coef_sh[1], kV = coef_sh[2];

    double sD = 0.0, sV = 0.0, sP = 0.0;
    Real* po = ca.phi[cur ^ 1];
    Real* qo = ca.pi[cur ^ 1];
    if (edge_blk)
      march_item<true, Real, Model, T>(g, po, qo, issue_next, slot, phase, raw, psi, bars, x0, y0, z0, nz, own_sm, halo_sm,
                                       cd, kD, kV, c0, c1, c2, c3, coef, sD, sV, sP);
    else
      march_item<false, Real, Model, T>(g, po, qo, issue_next, slot, phase, raw, psi, bars, x0, y0, z0, nz, own_sm, halo_sm,
                                        cd, kD, kV, c0, c1, c2, c3, coef, sD, sV, sP);
    double v[3] = {sD, sV, sP};
    block_reduce<3, NT>(v, red);

    // ---- stage tail = grid barrier.  Thread 0 publishes the block's partial sums (two sets of slots, by stage parity:
    // a block a stage ahead must not overwrite what a slower one still reads) and arrives (release: every store of this
    // block, fields included, is ordered before it by the block barrier + fence), then waits until every block has.
    // EVERY block then adds the partials in item order and advances its own copy of the scalars -- the same operations
    // on the same numbers in every block, so the same bits, with no second round trip through a "last" block; the next
    // stage's first loads go out before that, so their latency hides the reduction and the scalar update.
    const bool last_stage = k + 1 == sch.nstages;
    const double* part = g.partials + (size_t)(k & 1) * 3 * (size_t)g.nitems;
    if (tid == 0) {                                            // (the barrier inside block_reduce follows every thread's
      publish_partials(const_cast<double*>(part), (unsigned)g.nitems, (unsigned)item, v);   // last field store)
      __threadfence();
      atomicAdd(ca.release, 1u);
      if (!last_stage || blockIdx.x == 0) {
        const unsigned target = (unsigned)(k + 1) * gridDim.x;
        while (ld_acquire_u32(ca.release) < target) { }
        asm volatile("fence.proxy.async;" ::: "memory");       // other blocks' stores before this block's TMA loads
        if (!last_stage) issue_first(cur ^ 1);                 // at once: their latency hides the block barrier below,
      }                                                        // the reduction and the scalar update
    }
    if (last_stage && blockIdx.x != 0) break;                  // block 0 leaves the final scalars; the others are done
    __syncthreads();
    if (!last_stage) start_loads(cur ^ 1);
    double S3[3];
    block_sum_fixed3<NT>(part, (size_t)g.nitems, g.nitems, reinterpret_cast<double*>(psi), S3);   // psi planes: idle
    if (tid == 0) {
      const int i = sch.first + k;                             // stage index within the call
      StageLen len;
      len.dt = sch.dt; len.adaptive = sch.adaptive;
      len.w = sch.w[i % sch.ns];
      len.w_next = (!last_stage || !sch.call_ends) ? sch.w[(i + 1) % sch.ns] : 0.0;
      len.ends_step = (i % sch.ns) == sch.ns - 1;
      Scalars s = sc_sh;
      scalar_advance(s, g.tail.k, len, 1, S3[0], S3[1], S3[2]);
      sc_sh = s;
      coef_sh[0] = Real(s.c_drift); coef_sh[1] = Real(s.kD); coef_sh[2] = Real(s.kV);
      if (last_stage) *g.tail.sc = s;                          // block 0 only gets here
    }
    __syncthreads();
  }
}

}  // namespace pycool
