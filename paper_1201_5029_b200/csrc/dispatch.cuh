// dispatch.cuh -- <precision, model, tile> -> kernel template instance, and the launch code of each.
// Included by the per-model translation units (models_*.cu), which instantiate dispatch_one explicitly, so the
// instances of different models compile in parallel (build.py).  Internal.
#pragma once
#include "context.h"
#include "kick_tma.cuh"
#include "energy_tma.cuh"

namespace pycool {

using Tile0 = Tile<32, 8, 2>;
using Tile1 = Tile<32, 16, 2>;
using Tile2 = Tile<64, 8, 2>;
// kick_tma variants: <TX, TY, ring stages, rows per thread J, blocks per SM the registers are cut for>.
// (Tried and dropped, profiles/: ring of 4, 512-thread 2 x 1-site blocks, 64 x 32 tiles; for the Q-ball model a ring of
// 2 with three blocks per SM at 80 registers (620 bytes of spills): 384 us against 245 -- never faster.)
template <typename Real> using TTile3 = TmaTile<Real, 64, 16, 3, 2, sizeof(Real) == 4 ? 2 : 1>;   // 256 thr x (2 x 2 sites)
template <typename Real> using TTile4 = TmaTile<Real, 32, 16, 3, 2, 1>;   // 128 threads x (2 x 2 sites): small N
template <typename Real> using TTile5 = TmaTile<Real, 128, 8, 3, 2, sizeof(Real) == 4 ? 2 : 1>;   // 1 KB rows
template <typename Real> using TTile6 = TmaTile<Real, 128, 16, 3, 2, 1>;  // 512 threads: twice the bytes per plane (one field)
template <typename Real> using TTile7 = TmaTile<Real, 32, 16, 3, 1, 2>;   // 256 threads x (2 x 1 sites), two blocks per
template <typename Real> using TTile8 = TmaTile<Real, 64, 8, 3, 1, 2>;    //   SM: ALU-heavy models (Q-ball)
template <typename Real> using TTile9 = TmaTile<Real, 128, 16, 3, 4, 1>;   // 256 threads x (2 x 4 sites): one field
template <typename Real> using TTile10 = TmaTile<Real, 32, 16, 3, 1, 1>;   // 256 threads x (2 x 1 sites), full register
                                                                           //   file: three and four fp64 fields
// fp32 only: x quads (float4 accesses), 4 x 1 sites per thread, 256 threads, two blocks per SM -- the fp32 kernel is
// bound by its instruction count, and a quad needs 9 shared-memory loads for its 4 sites where 2 x 2 sites need 12
template <typename Real> using TTile11 = TmaTile<Real, 128, 8, 3, 1, 2, sizeof(Real) == 4 ? 4 : 2>;
// Q-ball, fp64: 32 x 8 tile, 128 threads x (2 x 1 sites), FOUR blocks per SM -- the same 16 warps per SM as variant 7,
// but four independent per-plane barriers instead of two, so the long finalise phase (the logarithm) of one block
// overlaps the load / drift phase of the others: 0.729 against 0.799 ms per step in one process (profiles/r2)
template <typename Real> using TTile12 = TmaTile<Real, 32, 8, 3, 1, 4>;
#define PYCOOL_TMA_TILES(X) \
  X(3, TTile3) X(4, TTile4) X(5, TTile5) X(6, TTile6) X(7, TTile7) X(8, TTile8) X(9, TTile9) X(10, TTile10) \
  X(11, TTile11) X(12, TTile12)

// Which <Real, Model, tile> instances are compiled at all: the ring must fit in shared memory, and the per-thread
// state (2 x J sites x NF fields x (A, B, two planes of phi', pi)) must fit the variant's register budget --
// instances that would spill are not built (pycool_set_tile answers PYCOOL_EINVAL for them).
template <typename Real, class Model, class T>
constexpr bool tile_built() {
  constexpr int NF = Model::NF;
  if (TmaSmem<Real, Model, T>::TOTAL > kMaxSmem) return false;
  if (T::TX == 128 && T::TY == 8 && T::J == 1 && T::XW == 2) return false;   // variant 11 exists as x quads (fp32) only
  if (T::MINB == 4 && !(std::is_same<Model, QBall>::value && sizeof(Real) == 8)) return false;   // variant 12: Q-ball only
  if (T::J == 4 && NF > 1) return false;                       // 2 x 4 sites per thread: one-field lattices only
  if (T::NT == 512 && NF > 2) return false;                    // 512 threads: 128 registers each
  if (T::MINB >= 2 && NF > 2) return false;                    // two blocks per SM: 128 registers each
  if (T::J == 2 && NF > 2 && sizeof(Real) == 8) return false;  // 2 x 2 sites x >= 3 fp64 fields: > 255 registers
  if (Model::kTestModel && (T::NT == 512 || (T::J == 1 && T::MINB == 2))) return false;   // the free test model gets
  return true;                                                 // the general-purpose variants only (library size)
}

// ---- kernel dispatch: <precision, model, nf, tile> -> template instance ----
template <typename Real, class Model, class T>
int launch_kick_t(pycool_ctx* c) {
  constexpr size_t smem = kick_smem_bytes<Real, Model, T>();
  if (c->resident[c->tile] < 0) {                              // once per context, i.e. per device
    CUDA_TRY(c, cudaFuncSetAttribute(kick_fused<Real, Model, T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)smem));
    c->resident[c->tile] = 2 * c->sms;                         // not persistent: a guess does
  }
  KickArgs<Real> g;
  g.phi_in = (const Real*)c->phi[c->cur];
  g.pi_in = (const Real*)c->pi[c->cur];
  g.phi_out = (Real*)c->phi[c->cur ^ 1];
  g.pi_out = (Real*)c->pi[c->cur ^ 1];
  g.sc = c->sc;
  g.partials = c->partials;
  g.tail.sc = c->sc;
  g.tail.ticket = c->ticket;
  g.tail.work = c->ticket + 1;
  g.tail.fused = c->fused_tail ? 1 : 0;
  g.tail.k = c->kc;
  g.tail.len = c->len;
  g.L = c->lay;
  g.zc = c->zc;
  g.c1 = c->c[1]; g.c2 = c->c[2]; g.c3 = c->c[3];
  g.mp = c->mp;
  kick_fused<Real, Model, T><<<c->grid, T::NT, smem, c->stream>>>(g);
  CUDA_TRY(c, cudaGetLastError());
  return PYCOOL_OK;
}
// Blocks of this kick_tma instance that fit on the device at once (0 on error, message in c->err); the first
// call also opts the instance in to its dynamic shared memory.
template <typename Real, class Model, class T>
int tma_resident(pycool_ctx* c, int tile_) {
  if (c->resident[tile_] >= 0) return c->resident[tile_];      // cached per context, i.e. per device
  constexpr size_t smem = TmaSmem<Real, Model, T>::TOTAL;
  int per_sm = 0;
  cudaError_t e = cudaFuncSetAttribute(kick_tma<Real, Model, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kick_tma<Real, Model, T>, T::NT, smem);
  if (e != cudaSuccess || per_sm * c->sms < 1) {
    fail(c, PYCOOL_ECUDA, "kick_tma does not fit on an SM (%zu bytes of shared memory): %s", smem, cudaGetErrorString(e));
    cudaGetLastError();
    return 0;
  }
  c->resident[tile_] = per_sm * c->sms;
  return c->resident[tile_];
}

template <typename Real, class Model, class T>
int launch_tma_t(pycool_ctx* c) {
  constexpr size_t smem = TmaSmem<Real, Model, T>::TOTAL;
  const int resident = tma_resident<Real, Model, T>(c, c->tile);
  if (resident < 1) return PYCOOL_ECUDA;
  TmaArgs<Real> g;
  g.phi_out = (Real*)c->phi[c->cur ^ 1];
  g.pi_out = (Real*)c->pi[c->cur ^ 1];
  g.sc = c->sc;
  g.partials = c->partials;
  g.tail.sc = c->sc;
  g.tail.ticket = c->ticket;
  g.tail.work = c->ticket + 1;
  g.tail.fused = c->fused_tail ? 1 : 0;
  g.tail.k = c->kc;
  g.tail.len = c->len;
  g.L = c->lay;
  g.zc = c->zc;
  g.nbx = (int)c->grid.x; g.nby = (int)c->grid.y;
  g.nitems = (int)(c->grid.x * c->grid.y * c->grid.z);
  g.ry = c->region[1];
  g.c1 = c->c[1]; g.c2 = c->c[2]; g.c3 = c->c[3];
  g.mp = c->mp;
  // persistent: one block per resident slot, every further item claimed from a device counter (kick_tma.cuh);
  // else one block per item
  const int nblocks = c->persistent && resident < g.nitems ? resident : g.nitems;
  c->blocks_launched = nblocks;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)nblocks);
  cfg.blockDim = dim3(T::NT);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = c->stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;    // see the kernel's griddepcontrol.wait
  attr[0].val.programmaticStreamSerializationAllowed = c->overlap_launch ? 1 : 0;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  CUDA_TRY(c, cudaLaunchKernelEx(&cfg, kick_tma<Real, Model, T>, c->tm[c->cur][0], c->tm[c->cur][1], g));
  return PYCOOL_OK;
}
// ---- small lattices: several stages per cooperative launch (kick_tma_coop), variants 3 and 4 only
template <class T> constexpr bool coop_tile() { return T::S == 3 && T::J == 2 && T::MINB == 1 && T::XW == 2 && T::TY == 16 && T::TX <= 64; }

// Co-resident blocks of kick_tma_coop on this device (0: no cooperative launch here).
template <typename Real, class Model, class T>
int coop_resident(pycool_ctx* c, int tile_) {
  if (c->coop_resident[tile_] >= 0) return c->coop_resident[tile_];
  constexpr size_t smem = TmaSmem<Real, Model, T>::TOTAL;
  int per_sm = 0, coop = 0;
  cudaError_t e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device);
  if (e == cudaSuccess && coop)
    e = cudaFuncSetAttribute(kick_tma_coop<Real, Model, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess && coop)
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kick_tma_coop<Real, Model, T>, T::NT, smem);
  if (e != cudaSuccess) { cudaGetLastError(); per_sm = 0; }
  c->coop_resident[tile_] = coop ? per_sm * c->sms : 0;
  return c->coop_resident[tile_];
}

// One cooperative launch of c->coop.nstages stages starting from buffer c->cur (the caller flips c->cur afterwards).
template <typename Real, class Model, class T>
int launch_tma_coop_t(pycool_ctx* c) {
  constexpr size_t smem = TmaSmem<Real, Model, T>::TOTAL;
  TmaArgs<Real> g;
  g.phi_out = nullptr; g.pi_out = nullptr;                    // per stage: CoopArgs
  g.sc = c->sc;
  g.partials = c->partials;
  g.tail.sc = c->sc;
  g.tail.ticket = c->ticket;
  g.tail.work = c->ticket + 1;
  g.tail.fused = 1;
  g.tail.k = c->kc;
  g.tail.len = c->len;
  g.L = c->lay;
  g.zc = c->zc;
  g.nbx = (int)c->grid.x; g.nby = (int)c->grid.y;
  g.nitems = (int)(c->grid.x * c->grid.y * c->grid.z);
  g.ry = c->region[1];
  g.c1 = c->c[1]; g.c2 = c->c[2]; g.c3 = c->c[3];
  g.mp = c->mp;
  CoopArgs<Real> ca;
  for (int b = 0; b < 2; ++b) { ca.phi[b] = (Real*)c->phi[b]; ca.pi[b] = (Real*)c->pi[b]; }
  ca.cur0 = c->cur;
  ca.release = c->ticket + 2;
  CUDA_TRY(c, cudaMemsetAsync(ca.release, 0, sizeof(unsigned int), c->stream));
  CoopSchedule sch = c->coop;
  void* args[] = {(void*)&c->tm[0][0], (void*)&c->tm[0][1], (void*)&c->tm[1][0], (void*)&c->tm[1][1], (void*)&g, (void*)&ca,
                  (void*)&sch};
  CUDA_TRY(c, cudaLaunchCooperativeKernel((const void*)kick_tma_coop<Real, Model, T>, dim3((unsigned)g.nitems), dim3(T::NT),
                                          args, smem, c->stream));
  c->blocks_launched = g.nitems;
  return PYCOOL_OK;
}

template <typename Real, class Model>
long long coop_m(pycool_ctx* c, Op op, int tile_) {
  switch (tile_) {
#define X(ID, TT)                                                                                             \
  case ID:                                                                                                    \
    if constexpr (coop_tile<TT<Real>>() && tile_built<Real, Model, TT<Real>>())                               \
      return op == OP_KICK_COOP ? launch_tma_coop_t<Real, Model, TT<Real>>(c) : coop_resident<Real, Model, TT<Real>>(c, tile_); \
    else return op == OP_KICK_COOP ? PYCOOL_EINVAL : 0;
    PYCOOL_TMA_TILES(X)
#undef X
    default: return op == OP_KICK_COOP ? PYCOOL_EINVAL : 0;
  }
}

template <typename Real, class Model>
int launch_kick_m(pycool_ctx* c) {
  const int tile_ = c->tile;
  switch (tile_) {
    case 0: return launch_kick_t<Real, Model, Tile0>(c);
    case 1: return launch_kick_t<Real, Model, Tile1>(c);
    case 2: return launch_kick_t<Real, Model, Tile2>(c);
#define X(ID, TT)                                                                                           \
  case ID:                                                                                                  \
    if constexpr (tile_built<Real, Model, TT<Real>>()) return launch_tma_t<Real, Model, TT<Real>>(c);       \
    else return fail(c, PYCOOL_EINVAL, "kernel variant %d is not built for this model and precision", ID);
    PYCOOL_TMA_TILES(X)
#undef X
    default: return 0;
  }
}
template <typename Real, class Model>
size_t kick_smem_m(int tile_) {
  switch (tile_) {
    case 0: return kick_smem_bytes<Real, Model, Tile0>();
    case 1: return kick_smem_bytes<Real, Model, Tile1>();
    case 2: return kick_smem_bytes<Real, Model, Tile2>();
#define X(ID, TT) case ID: return TmaSmem<Real, Model, TT<Real>>::TOTAL;
    PYCOOL_TMA_TILES(X)
#undef X
    default: return 0;
  }
}
template <typename Real, class Model>
bool tile_built_m(int tile_) {
  switch (tile_) {
    case 0: case 1: case 2: return true;
#define X(ID, TT) case ID: return tile_built<Real, Model, TT<Real>>();
    PYCOOL_TMA_TILES(X)
#undef X
    default: return false;
  }
}
template <typename Real, class Model>
int kick_resident_m(pycool_ctx* c, int tile_) {
  switch (tile_) {
    case 0: case 1: case 2: return 2 * c->sms;          // register-prefetch kernel: not persistent, a guess does
#define X(ID, TT)                                                                                            \
  case ID:                                                                                                   \
    if constexpr (tile_built<Real, Model, TT<Real>>()) return tma_resident<Real, Model, TT<Real>>(c, tile_); \
    else return 0;
    PYCOOL_TMA_TILES(X)
#undef X
    default: return 0;
  }
}
// TMA-fed energy sums (energy_tma.cuh): ghost layout, at most two fields (the ring of more does not fit).
template <typename Real, class Model, class T>
int launch_energy_tma(pycool_ctx* c) {
  constexpr size_t smem = EnergySmem<Real, Model, T>::TOTAL;
  bool& attr_done = c->energy_attr[T::TX == 64 ? 0 : (T::J == 1 ? 1 : 2)];   // per context, i.e. per device
  if (!attr_done) {
    CUDA_TRY(c, cudaFuncSetAttribute(energy_tma<Real, Model, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_done = true;
  }
  CUtensorMap tm_phi, tm_pi;
  if (int st = encode_one(c, c->phi[c->cur], T::TX, T::TY, &tm_phi)) return st;
  if (int st = encode_one(c, c->pi[c->cur], T::TX, T::TY, &tm_pi)) return st;
  EnergyArgs<Real> g;
  g.phi = (const Real*)c->phi[c->cur];
  g.pi = (const Real*)c->pi[c->cur];
  g.sc = c->energy_through_drift ? c->sc : nullptr;
  g.partials = c->partials;
  g.L = c->lay;
  g.zc = c->N < 32 ? c->N : 32;
  g.nbx = (c->N + T::TX - 1) / T::TX;
  g.nby = (c->N + T::TY - 1) / T::TY;
  g.c1 = c->c[1]; g.c2 = c->c[2]; g.c3 = c->c[3];
  g.mp = c->mp;
  const size_t nb = (size_t)g.nbx * g.nby * ((c->N + g.zc - 1) / g.zc);
  if ((3 * (size_t)Model::NF + 1) * nb > c->partials_cap) return -1;       // caller falls back
  energy_tma<Real, Model, T><<<(unsigned)nb, T::NT, smem, c->stream>>>(tm_phi, tm_pi, g);
  CUDA_TRY(c, cudaGetLastError());
  c->energy_nb = (int)nb;
  return PYCOOL_OK;
}
template <typename Real, class Model>
int launch_energy_m(pycool_ctx* c, int nb) {
  if constexpr (Model::NF <= 2) {
    if (c->lay.gx > 0 && c->energy_tma) {
      // automatic: two fp64 fields above N = 64 take the 32 x 16 tile with 2 x 1 sites per thread, two blocks per SM
      // (16 warps); fp32 fields, one-field lattices and small lattices the 128-thread 32 x 16 tile with 2 x 2 sites
      // (measured at 512^3 fp32: 0.74 against 0.86 ms; oscillon 256^3: 0.099 against 0.121 ms); 2: 64 x 16, 2 x 2 sites
      const bool light = sizeof(Real) == 4 || Model::NF == 1 || c->N <= 64;
      const int v = c->energy_tma == 1 ? (light ? 4 : 3) : c->energy_tma;
      const int st = v == 2 ? launch_energy_tma<Real, Model, TmaTile<Real, 64, 16, 3, 2, 1>>(c)
                   : v == 3 ? launch_energy_tma<Real, Model, TTile7<Real>>(c)
                            : launch_energy_tma<Real, Model, TTile4<Real>>(c);
      if (st >= 0) return st;
    }
  }
  energy_sums<Real, Model><<<nb, 256, 0, c->stream>>>((const Real*)c->phi[c->cur], (const Real*)c->pi[c->cur],
                                                      c->lay, c->c[1], c->c[2], c->c[3], c->mp, c->partials,
                                                      c->energy_through_drift ? c->sc : nullptr);
  CUDA_TRY(c, cudaGetLastError());
  c->energy_nb = nb;
  return PYCOOL_OK;
}

template <typename Real, class Model>
long long dispatch_one(pycool_ctx* c, Op op, int arg) {
  if (op == OP_KICK) return launch_kick_m<Real, Model>(c);
  if (op == OP_KICK_COOP) return coop_m<Real, Model>(c, op, c->tile);
  if (op == OP_COOP_RESIDENT) return coop_m<Real, Model>(c, op, arg);
  if (op == OP_ENERGY) return launch_energy_m<Real, Model>(c, arg);
  if (op == OP_RESIDENT) return kick_resident_m<Real, Model>(c, arg);
  if (op == OP_BUILT) return tile_built_m<Real, Model>(arg) ? 1 : 0;
  return (long long)kick_smem_m<Real, Model>(arg);
}

#define PYCOOL_INSTANTIATE_MODEL(M)                                          \
  template long long dispatch_one<double, M>(pycool_ctx*, Op, int);          \
  template long long dispatch_one<float, M>(pycool_ctx*, Op, int);

}  // namespace pycool
