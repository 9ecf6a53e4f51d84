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
  sc->a = a;
  if (set_pa) sc->p_a = p_a;
}

}  // namespace pycool
