// potentials.cuh -- per-model potentials V(phi_1..phi_nf) and dV/dphi_f as C++ template instances.
//
// Replaces PyCOOL's run-time textual code generation (jinja2/SymPy -> CUDA source): each
// model is a struct with a static, fully inlined `eval`, so the kick kernel is compiled once per
// <Real, Model> pair with the potential folded into its finalize step.
//
// Models (the paper prints V only; the derivatives are spelled out here):
//   Free<NF>   V = sum_f 1/2 m_f^2 phi_f^2                                      (test model)
//   Chaotic    V = 1/2 m^2 phi^2 + 1/2 g^2 phi^2 chi^2                          (3.2) PAPER.md:427
//   Oscillon   V = 1/2 m^2 phi^2 - lambda/4 phi^4 + g6/6 phi^6                  (3.3) PAPER.md:456 (reading G6)
//   QBall      V = m^2 r2 (1 + K ln(r2/M^2)) + lambda6 r2^3/mpl^2, r2 = (phi1^2+phi2^2)/2
//                                                                               (3.4) PAPER.md:481 (G6-G8)
#pragma once
#include <cfloat>
#include <cstring>

namespace pycool {

struct ModelParams {
  double p[8];       // as in pycool_params.p
  double inv_mpl2;   // 1/mpl^2 (0 for a static background)
};

template <typename T> __device__ __forceinline__ T min_normal();
template <> __device__ __forceinline__ double min_normal<double>() { return DBL_MIN; }
template <> __device__ __forceinline__ float min_normal<float>() { return FLT_MIN; }

// Natural logarithm of a positive finite double, for the Q-ball potential (3.4).  CUDA's log() costs ~150
// instructions per call in this kernel (slow-path branches, integer work), which made the Q-ball kick ALU-bound;
// this one is ~40: x = 2^e m with m in [sqrt(1/2), sqrt(2)), s = (m-1)/(m+1), ln m = 2 s sum_k s^(2k)/(2k+1)
// (|s| <= 0.1716, 11 terms: truncation 2e-19), ln x = e ln2_hi + (e ln2_lo + ln m) with the two-part ln 2 of
// fdlibm.  Error <= 2.1 ulp against logl over [1e-300, 1e300], near 1 and at the sqrt 2 switch
// (tests/test_abi_cpu.py compiles this very function for the host, tests/log_pos_check.cu, and checks it).
__host__ __device__ __forceinline__ double log_pos(double x) {
  int e = 0;
  if (x < 2.2250738585072014e-308) { x *= 18014398509481984.0; e = -54; }      // subnormal: scale by 2^54
#if defined(__CUDA_ARCH__)
  int hi = __double2hiint(x);
  const int lo = __double2loint(x);
#else
  unsigned long long bits;
  memcpy(&bits, &x, sizeof bits);
  int hi = (int)(bits >> 32);
  const int lo = (int)(unsigned)(bits & 0xffffffffu);
#endif
  e += (hi >> 20) - 1023;
  hi = (hi & 0x000fffff) | 0x3ff00000;                                           // m in [1, 2)
  if (hi >= 0x3ff6a09e) { hi -= 0x00100000; e += 1; }                            // m >= ~sqrt 2: halve it
#if defined(__CUDA_ARCH__)
  const double m = __hiloint2double(hi, lo);
#else
  bits = ((unsigned long long)(unsigned)hi << 32) | (unsigned)lo;
  double m;
  memcpy(&m, &bits, sizeof m);
#endif
  // s = (m - 1)/(m + 1) without the compiler's division (its slow-path test costs a divergent call per site):
  // r ~ 1/d from the hardware's seed (>= 20 bits; a float reciprocal on the host), one Newton step (2^-40), then one
  // correction of the quotient (error 2^-40 x 2^-40) -- within 1 ulp; d = m + 1 is in [1.7, 2.42), nothing can overflow
  const double d = m + 1.0, n = m - 1.0;
#if defined(__CUDA_ARCH__)
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
#else
  double r = (double)(1.0f / (float)d);
#endif
  r = fma(fma(-d, r, 1.0), r, r);
  double s = n * r;
  s = fma(fma(-d, s, n), r, s);
  const double z = s * s;
  // sum_{k=0..10} z^k / (2k + 3), Estrin's scheme: 5 dependent operations instead of Horner's 11 (the kick
  // has two of these chains per thread in flight and few warps to hide them behind)
  const double z2 = z * z, z4 = z2 * z2, z8 = z4 * z4;
  const double a0 = fma(1.0 / 5.0, z, 1.0 / 3.0), a1 = fma(1.0 / 9.0, z, 1.0 / 7.0);
  const double a2 = fma(1.0 / 13.0, z, 1.0 / 11.0), a3 = fma(1.0 / 17.0, z, 1.0 / 15.0);
  const double a4 = fma(1.0 / 21.0, z, 1.0 / 19.0), a5 = 1.0 / 23.0;
  const double b0 = fma(a1, z2, a0), b1 = fma(a3, z2, a2), b2 = fma(a5, z2, a4);
  const double p = fma(b2, z8, fma(b1, z4, b0));
  const double two_s = s + s;
  const double lnm = fma(two_s * z, p, two_s);                                   // 2 s (1 + z p)
  const double de = (double)e;
  return fma(de, 6.93147180369123816490e-01, fma(de, 1.90821492927058770002e-10, lnm));
}

__device__ __forceinline__ double log_of(double x) { return log_pos(x); }
__device__ __forceinline__ float log_of(float x) { return logf(x); }

// Coefficients are converted to the compute type T once per thread (Coef), then eval() is pure T arithmetic.
template <int NF_>
struct Free {
  static constexpr int NF = NF_;
  static constexpr bool kTestModel = true;
  template <typename T> struct Coef {
    T m2[NF_];
    __device__ explicit Coef(const ModelParams& mp) {
#pragma unroll
      for (int f = 0; f < NF_; ++f) m2[f] = T(mp.p[f]);
    }
  };
  template <typename T>
  static __device__ __forceinline__ T eval(const Coef<T>& c, const T* phi, T* dV) {
    T v = T(0);
#pragma unroll
    for (int f = 0; f < NF_; ++f) {
      dV[f] = c.m2[f] * phi[f];
      v += T(0.5) * dV[f] * phi[f];
    }
    return v;
  }
};

struct Chaotic {
  static constexpr int NF = 2;
  static constexpr bool kTestModel = false;
  template <typename T> struct Coef {
    T m2, g2;
    __device__ explicit Coef(const ModelParams& mp) : m2(T(mp.p[0])), g2(T(mp.p[1])) {}
  };
  template <typename T>
  static __device__ __forceinline__ T eval(const Coef<T>& c, const T* phi, T* dV) {
    const T ph = phi[0], ch = phi[1];
    const T ph2 = ph * ph;
    const T u = c.m2 + c.g2 * (ch * ch);   // m^2 + g^2 chi^2
    dV[0] = ph * u;                        // m^2 phi + g^2 phi chi^2
    dV[1] = c.g2 * ph2 * ch;               // g^2 phi^2 chi
    return T(0.5) * ph2 * u;
  }
};

struct Oscillon {
  static constexpr int NF = 1;
  static constexpr bool kTestModel = false;
  template <typename T> struct Coef {
    T m2, lam, g6, hm2, ql, sg;
    __device__ explicit Coef(const ModelParams& mp)
        : m2(T(mp.p[0])), lam(T(mp.p[1])), g6(T(mp.p[2])), hm2(T(0.5 * mp.p[0])), ql(T(mp.p[1] / 4.0)),
          sg(T(mp.p[2] / 6.0)) {}
  };
  template <typename T>
  static __device__ __forceinline__ T eval(const Coef<T>& c, const T* phi, T* dV) {
    const T ph = phi[0], p2 = ph * ph;
    dV[0] = ph * (c.m2 + p2 * (c.g6 * p2 - c.lam));       // m^2 phi - lambda phi^3 + g6 phi^5
    return p2 * (c.hm2 + p2 * (c.sg * p2 - c.ql));
  }
};

struct QBall {
  static constexpr int NF = 2;
  static constexpr bool kTestModel = false;
  template <typename T> struct Coef {
    T m2, K, invM2, six;
    __device__ explicit Coef(const ModelParams& mp)
        : m2(T(mp.p[0])), K(T(mp.p[1])), invM2(T(1.0 / mp.p[2])), six(T(mp.p[3] * mp.inv_mpl2)) {}
  };
  template <typename T>
  static __device__ __forceinline__ T eval(const Coef<T>& c, const T* phi, T* dV) {
    const T r2 = T(0.5) * (phi[0] * phi[0] + phi[1] * phi[1]);      // |Phi|^2, Phi = (phi1 + i phi2)/sqrt 2
    const T lg = (r2 < min_normal<T>()) ? T(0) : log_of(r2 * c.invM2);   // reading G8
    const T klg = c.K * lg;
    const T r4 = r2 * r2;
    const T common = c.m2 * (T(1) + c.K + klg) + T(3) * c.six * r4;
    dV[0] = common * phi[0];
    dV[1] = common * phi[1];
    return c.m2 * r2 * (T(1) + klg) + c.six * r4 * r2;
  }
};

}  // namespace pycool
