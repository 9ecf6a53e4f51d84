// cufft_api.h -- cuFFT loaded on first use (dlopen), not linked: a library FFT is a step the scope allows
// (initial conditions, spectra, the linearised solver's transforms); loading it lazily keeps the hot path free of
// it and lets the calls that need it fail loudly when it is missing.  Internal.
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>      // types only

namespace pycool {

struct CufftApi {
  cufftResult (*plan3d)(cufftHandle*, int, int, int, cufftType) = nullptr;
  cufftResult (*set_stream)(cufftHandle, cudaStream_t) = nullptr;
  cufftResult (*exec_z2d)(cufftHandle, cufftDoubleComplex*, cufftDoubleReal*) = nullptr;
  cufftResult (*exec_d2z)(cufftHandle, cufftDoubleReal*, cufftDoubleComplex*) = nullptr;
  cufftResult (*destroy)(cufftHandle) = nullptr;
  bool ok = false;
};
const CufftApi& cufft_api();   // defined in pycool.cu

}  // namespace pycool
