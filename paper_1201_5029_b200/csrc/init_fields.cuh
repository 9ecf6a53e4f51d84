// init_fields.cuh -- seeded Gaussian initial conditions on the device (reading G21).
//
// The paper takes its initial fluctuations from Defrost's generator without describing it, so the
// recipe is this repository's: per array a Gaussian random field with spectrum A(k) = amp (k^2 + m2)^q (k <= kmax),
//   F_j = A(k) (g1 + i g2)/sqrt 2,  (g1, g2) = Box-Muller of Philox4x32-10(counter = (j, array id), key = seed),
// Hermitian on the planes ix = 0 and ix = N/2, field = mean + sqrt 2 / L^1.5 sum_k F_k exp(+2 pi i n.x/N).
// fill_spectrum writes the half-spectrum (one thread per mode, counter-based: no state, any launch shape gives the
// same numbers), cuFFT does the inverse transform in place (Z2D, always double), scatter_real writes the result
// into the padded state layout with its ghost images.  Removes the host FFT and the PCIe upload at 1024^3.
#pragma once
#include <cstdint>

#include "kernels.cuh"

namespace pycool {

struct Spectrum { double mean, amp, m2, q, kmax; };

struct Philox4 { uint32_t w[4]; };

// Philox4x32 with 10 rounds (Salmon, Moraes, Dror, Shaw, SC'11).
__device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                                 uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
  }
  return Philox4{{c0, c1, c2, c3}};
}

// (g1, g2) of mode j of array `aid`: Box-Muller on two 32-bit uniforms (u = (w + 1/2) 2^-32, never 0 or 1)
__device__ __forceinline__ double2 mode_gaussians(unsigned long long j, uint32_t aid, unsigned long long seed) {
  const Philox4 p = philox4x32_10((uint32_t)j, (uint32_t)(j >> 32), aid, 0u, (uint32_t)seed, (uint32_t)(seed >> 32));
  const double u1 = ((double)p.w[0] + 0.5) * 2.3283064365386963e-10;     // 2^-32
  const double u2 = ((double)p.w[1] + 0.5) * 2.3283064365386963e-10;
  const double r = sqrt(-2.0 * log(u1));
  double s, c;
  sincospi(2.0 * u2, &s, &c);
  return double2{r * c, r * s};
}

// Half-spectrum F[iz][iy][ix], ix = 0 .. N/2, of one array.  One thread per mode.
__global__ void __launch_bounds__(256)
fill_spectrum(double2* __restrict__ F, int N, double L, Spectrum sp, uint32_t aid, unsigned long long seed) {
  const int H = N / 2 + 1;
  const unsigned long long nmodes = (unsigned long long)N * N * H;
  const double kf = 6.283185307179586476925 / L;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; j < nmodes; j += stride) {
    const int ix = (int)(j % H);
    const unsigned long long zy = j / H;
    const int iy = (int)(zy % N), iz = (int)(zy / N);
    const int nz = iz <= N / 2 ? iz : iz - N, ny = iy <= N / 2 ? iy : iy - N;
    const long long n2 = (long long)nz * nz + (long long)ny * ny + (long long)ix * ix;
    const double k = kf * sqrt((double)n2);
    double A = 0.0;
    if (n2 > 0 && !(sp.kmax > 0.0 && k > sp.kmax)) A = sp.amp * pow(k * k + sp.m2, sp.q);
    double2 f;
    const bool edge = ix == 0 || ix == N / 2;
    const int mz = (N - iz) % N, my = (N - iy) % N;              // mirror image under k -> -k within the plane
    if (edge && mz == iz && my == iy) {                          // self-conjugate mode: real
      const double2 g = mode_gaussians(j, aid, seed);
      f = double2{A * g.x, 0.0};
    } else if (edge && (long long)iz * N + iy > (long long)mz * N + my) {   // the later one of a mirror pair
      const unsigned long long jm = ((unsigned long long)mz * N + my) * H + ix;
      const double2 g = mode_gaussians(jm, aid, seed);
      f = double2{A * g.x * 0.70710678118654752440, -(A * g.y * 0.70710678118654752440)};
    } else {
      const double2 g = mode_gaussians(j, aid, seed);
      f = double2{A * g.x * 0.70710678118654752440, A * g.y * 0.70710678118654752440};
    }
    F[j] = f;
  }
}

// dst(f-th array of the padded state, with ghost images) = mean + scale * src, src = the in-place C2R result:
// [z][y][2 (N/2 + 1)] doubles, the first N of each row valid.
template <typename Real>
__global__ void __launch_bounds__(256)
scatter_real(Real* __restrict__ dst, Layout L, const double* __restrict__ src, double mean, double scale) {
  const int N = L.N;
  const size_t rp = 2 * (size_t)(N / 2 + 1);
  const size_t V = (size_t)N * N * N;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += stride) {
    const int x = (int)(i % N), y = (int)((i / N) % N), z = (int)(i / ((size_t)N * N));
    const double v = fma(scale, src[((size_t)z * N + y) * rp + x], mean);
    store_site<Real>(dst + (size_t)z * L.plane, L, x, y, (Real)v);
  }
}

// ------------------------------------------------------------------------------------------------ shell spectrum
// SURVEY.md 8(f) rank 3 (reading G22).  gather_real copies one array of the padded state into the
// in-place R2C layout [z][y][2 (N/2 + 1)] as doubles, cuFFT transforms it (D2Z), bin_shells adds w |F_k|^2 into the
// shell round(|n|) (w = 2 for the modes the half-spectrum stores once for a conjugate pair, 1 on the planes ix = 0
// and ix = N/2), F_k = norm * (D2Z output).  Per-block shared-memory histograms (atomics: the order of the adds
// inside a block is not fixed, so the last bits may differ from run to run -- a diagnostic, not part of the step),
// then reduce_shells adds the per-block rows in block order.
template <typename Real>
__global__ void __launch_bounds__(256)
gather_real(double* __restrict__ dst, const Real* __restrict__ src, Layout L) {
  const int N = L.N;
  const size_t rp = 2 * (size_t)(N / 2 + 1);
  const size_t V = (size_t)N * N * N;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += stride) {
    const int x = (int)(i % N), y = (int)((i / N) % N), z = (int)(i / ((size_t)N * N));
    dst[((size_t)z * N + y) * rp + x] = (double)src[L.at(0, z, y, x)];
  }
}

__global__ void __launch_bounds__(256)
bin_shells(const double2* __restrict__ F, int N, double norm2, int nbins, double* __restrict__ part /* [grid][2 nbins] */) {
  extern __shared__ double hist[];                             // [nbins] power, [nbins] counts
  for (int i = threadIdx.x; i < 2 * nbins; i += blockDim.x) hist[i] = 0.0;
  __syncthreads();
  const int H = N / 2 + 1;
  const unsigned long long nmodes = (unsigned long long)N * N * H;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; j < nmodes; j += stride) {
    const int ix = (int)(j % H);
    const unsigned long long zy = j / H;
    const int iy = (int)(zy % N), iz = (int)(zy / N);
    const int nz = iz <= N / 2 ? iz : iz - N, ny = iy <= N / 2 ? iy : iy - N;
    const long long n2 = (long long)nz * nz + (long long)ny * ny + (long long)ix * ix;
    const int shell = (int)floor(sqrt((double)n2) + 0.5);
    if (shell >= nbins) continue;
    const double w = (ix == 0 || (N % 2 == 0 && ix == N / 2)) ? 1.0 : 2.0;
    const double2 f = F[j];
    atomicAdd(&hist[shell], w * norm2 * fma(f.x, f.x, f.y * f.y));
    atomicAdd(&hist[nbins + shell], w);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 2 * nbins; i += blockDim.x) part[(size_t)blockIdx.x * 2 * nbins + i] = hist[i];
}

// Number- and energy-density spectra of one field (reading G24): with F^phi_k, F^pi_k
// the D2Z transforms scaled by norm = L^1.5 / (sqrt 2 N^3), u = a F^phi, v = F^pi / a,
//   w_k^2 = k_eff^2(n)/dx^2 + a^2 m_eff^2,  -k_eff^2 = eigenvalue of the stencil (2.7) on the mode,
//   n_k = 1/2 (w |u|^2 + |v|^2 / w)  (0 where w^2 <= 0),   rho_k = 1/2 (|v|^2 + w^2 |u|^2),
// added into the shell round(|n|) with the half-spectrum weight (2, or 1 on the planes ix = 0 and ix = N/2).
// hist: [nbins] number, [nbins] energy, [nbins] counts.
struct ModeSpectrumArgs {
  double norm2, a2, m_eff2, inv_dx2, c0, c1, c2, c3;
};
__global__ void __launch_bounds__(256)
bin_mode_spectra(const double2* __restrict__ Fphi, const double2* __restrict__ Fpi, int N, ModeSpectrumArgs g,
                 int nbins, double* __restrict__ part /* [grid][3 nbins] */) {
  extern __shared__ double hist[];
  for (int i = threadIdx.x; i < 3 * nbins; i += blockDim.x) hist[i] = 0.0;
  __syncthreads();
  const int H = N / 2 + 1;
  const unsigned long long nmodes = (unsigned long long)N * N * H;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  const double inv_n = 2.0 / (double)N;
  for (unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; j < nmodes; j += stride) {
    const int ix = (int)(j % H);
    const unsigned long long zy = j / H;
    const int iy = (int)(zy % N), iz = (int)(zy / N);
    const int nz = iz <= N / 2 ? iz : iz - N, ny = iy <= N / 2 ? iy : iy - N;
    const long long n2 = (long long)nz * nz + (long long)ny * ny + (long long)ix * ix;
    const int shell = (int)floor(sqrt((double)n2) + 0.5);
    if (shell >= nbins) continue;
    const double Cx = cospi(inv_n * ix), Cy = cospi(inv_n * iy), Cz = cospi(inv_n * iz);
    const double keff2 = -(g.c0 + 2.0 * g.c1 * (Cx + Cy + Cz) + 4.0 * g.c2 * (Cx * Cy + Cy * Cz + Cz * Cx) +
                           8.0 * g.c3 * Cx * Cy * Cz);
    const double w2 = keff2 * g.inv_dx2 + g.a2 * g.m_eff2;
    const double2 fp = Fphi[j], fq = Fpi[j];
    const double u2 = g.norm2 * g.a2 * fma(fp.x, fp.x, fp.y * fp.y);
    const double v2 = g.norm2 * fma(fq.x, fq.x, fq.y * fq.y) / g.a2;
    const double wgt = (ix == 0 || (N % 2 == 0 && ix == N / 2)) ? 1.0 : 2.0;
    const double rho = 0.5 * (v2 + w2 * u2);
    double num = 0.0;
    if (w2 > 0.0) {
      const double w = sqrt(w2);
      num = 0.5 * (w * u2 + v2 / w);
    }
    atomicAdd(&hist[shell], wgt * num);
    atomicAdd(&hist[nbins + shell], wgt * rho);
    atomicAdd(&hist[2 * nbins + shell], wgt);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 3 * nbins; i += blockDim.x) part[(size_t)blockIdx.x * 3 * nbins + i] = hist[i];
}

__global__ void __launch_bounds__(256) reduce_shells(const double* __restrict__ part, int nblocks, int n, double* __restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double s = 0.0;
  for (int b = 0; b < nblocks; ++b) s += part[(size_t)b * n + i];
  out[i] = s;
}

}  // namespace pycool
