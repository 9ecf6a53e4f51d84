// linear.cu -- context, launch sequencing and the C ABI of the linearised solver (include/pycool_linear.h).
//
// One pycool_linear_step(n, GROWTH) call enqueues, on the context's stream and without a host synchronisation:
//     lin_background   (1 thread)   background through n x stages(order) stages + the per-stage coefficient table
//     lin_growth       (thread per class x column)   growth matrices M(n dt, k_eff^2) of (2.51)
//     lin_apply        (thread per mode x pair of rows of M)   every Fourier mode multiplied by its class's matrix
// and with NAIVE: lin_background, then lin_naive (thread per mode through every stage).  Kernels: linear.cuh.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>

#include <cuda_runtime.h>

#include "../../include/pycool_linear.h"
#include "cufft_api.h"
#include "linear.cuh"

using namespace pycool;

struct pycool_linear_ctx {
  int N = 0, nf = 0, order = 0, nstages = 0, device = 0, sms = 0;
  double L = 0, dt = 0;
  size_t nmodes = 0, V = 0;
  unsigned nclasses = 0;
  LinConst k{};
  LinStencil sc{};
  double w[16];
  cudaStream_t stream = nullptr;
  LinBackground* bg = nullptr;      // device
  LinEnergyOut* en = nullptr;       // device
  double* d_w = nullptr;            // device: stage weights
  double2* dPhi = nullptr;          // device: [nf][nmodes]
  double2* dPi = nullptr;
  double* M = nullptr;              // device: [nclasses][2 nf][2 nf]
  void* table = nullptr;            // device: LinStage<nf>[table_cap]
  size_t table_cap = 0;
  bool have_growth = false;
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  int last_method = -1;
  std::string err;
};

namespace {

thread_local std::string g_lin_create_err = "no error";

int lfail(pycool_linear_ctx* c, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (c) c->err = buf; else g_lin_create_err = buf;
  return code;
}
#define LIN_TRY(c, expr)                                                                            \
  do {                                                                                              \
    cudaError_t e_ = (expr);                                                                        \
    if (e_ != cudaSuccess) return lfail((c), PYCOOL_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

struct OnDev {                      // run on the context's device, restore the caller's
  int prev = -1;
  explicit OnDev(const pycool_linear_ctx* c) {
    int cur = -1;
    if (c && cudaGetDevice(&cur) == cudaSuccess && cur != c->device) { prev = cur; cudaSetDevice(c->device); }
  }
  ~OnDev() { if (prev >= 0) cudaSetDevice(prev); }
};

int stage_weights(int order, double* w) {
  double tmp[16];
  const int s = pycool_stage_weights(order, tmp, 16);   // (2.42)-(2.45), Table 1: one table for both solvers
  for (int i = 0; i < s; ++i) w[i] = tmp[i];
  return s;
}

size_t stage_bytes(int nf) { return (size_t)(2 + nf * nf) * sizeof(double); }

int ensure_table(pycool_linear_ctx* c, size_t nst) {
  if (nst <= c->table_cap) return PYCOOL_OK;
  if (c->table) { cudaStreamSynchronize(c->stream); cudaFree(c->table); c->table = nullptr; c->table_cap = 0; }
  if (cudaMalloc(&c->table, nst * stage_bytes(c->nf)) != cudaSuccess) {
    cudaGetLastError();
    return lfail(c, PYCOOL_ENOMEM, "cudaMalloc of the stage table (%zu stages) failed", nst);
  }
  c->table_cap = nst;
  return PYCOOL_OK;
}

template <int NF>
int step_t(pycool_linear_ctx* c, int nsteps, int method) {
  const size_t nst = (size_t)nsteps * c->nstages;
  if (int st = ensure_table(c, nst)) return st;
  LinStage<NF>* table = (LinStage<NF>*)c->table;
  const size_t plane = (size_t)c->N * (c->N / 2 + 1);          // modes of one i_z plane: the x extent of the mode grids
  LIN_TRY(c, cudaEventRecord(c->ev[0], c->stream));
  lin_background<NF><<<1, 1, 0, c->stream>>>(c->bg, c->k, c->d_w, c->nstages, nsteps, c->dt, table);
  LIN_TRY(c, cudaGetLastError());
  LIN_TRY(c, cudaEventRecord(c->ev[1], c->stream));
  if (method == PYCOOL_LINEAR_GROWTH) {
    const unsigned long long nthreads = (unsigned long long)c->nclasses * 2 * NF;
    lin_growth<NF><<<(unsigned)((nthreads + kLinThreads - 1) / kLinThreads), kLinThreads, 0, c->stream>>>(
        table, nst, c->sc, c->N, c->nclasses, c->M);
    LIN_TRY(c, cudaGetLastError());
    LIN_TRY(c, cudaEventRecord(c->ev[2], c->stream));
    using Apply = LinApplyCfg<NF, kLinApplyRows>;
    lin_apply<NF, kLinApplyRows><<<dim3((unsigned)((plane + Apply::MPB - 1) / Apply::MPB), (unsigned)c->N), Apply::NT, 0,
                                   c->stream>>>(c->dPhi, c->dPi, c->M, c->N, c->nmodes);
    LIN_TRY(c, cudaGetLastError());
    c->have_growth = true;
  } else {
    LIN_TRY(c, cudaEventRecord(c->ev[2], c->stream));
    lin_naive<NF><<<dim3((unsigned)((plane + kLinThreads - 1) / kLinThreads), (unsigned)c->N), kLinThreads, 0, c->stream>>>(
        c->dPhi, c->dPi, table, nst, c->sc, c->N, c->nmodes);
    LIN_TRY(c, cudaGetLastError());
  }
  LIN_TRY(c, cudaEventRecord(c->ev[3], c->stream));
  c->last_method = method;
  return PYCOOL_OK;
}

void destroy(pycool_linear_ctx* c) {
  if (c->stream) cudaStreamSynchronize(c->stream);
  for (cudaEvent_t e : c->ev) if (e) cudaEventDestroy(e);
  for (void* p : {(void*)c->bg, (void*)c->en, (void*)c->d_w, (void*)c->dPhi, (void*)c->dPi, (void*)c->M, c->table})
    if (p) cudaFree(p);
  if (c->stream) cudaStreamDestroy(c->stream);
  delete c;
}

}  // namespace

// =================================================================================================== C ABI
extern "C" {

size_t pycool_linear_num_classes(int N) {
  if (N < 3 || N > 2048) return 0;
  const unsigned long long M = (unsigned long long)(N / 2);
  return (size_t)((M + 1) * (M + 2) * (M + 3) / 6);
}

int pycool_linear_create(pycool_linear_ctx** out, int N, double L, int nf, const pycool_params* p, int order,
                         double dt) {
  if (!out) return lfail(nullptr, PYCOOL_EINVAL, "out is NULL");
  *out = nullptr;
  if (!p) return lfail(nullptr, PYCOOL_EINVAL, "params is NULL");
  if (N < 3 || N > 2048 || nf < 1 || nf > kLinMaxNF) return lfail(nullptr, PYCOOL_EINVAL, "N must be 3..2048, nfields 1..4");
  if (p->precision != 0 && p->precision != 64) return lfail(nullptr, PYCOOL_EINVAL, "the linearised solver is double precision only");
  if (!(L > 0) || !std::isfinite(L)) return lfail(nullptr, PYCOOL_EINVAL, "L must be finite and > 0");
  double w[16];
  const int ns = stage_weights(order, w);
  if (ns == 0) return lfail(nullptr, PYCOOL_EINVAL, "order must be 2, 4, 6 or 8");
  if (dt == 0 || !std::isfinite(dt)) return lfail(nullptr, PYCOOL_EINVAL, "dt must be finite and non-zero");
  if (p->model < PYCOOL_FREE || p->model > PYCOOL_QBALL) return lfail(nullptr, PYCOOL_EINVAL, "unknown model");
  if ((p->model == PYCOOL_CHAOTIC || p->model == PYCOOL_QBALL) && nf != 2)
    return lfail(nullptr, PYCOOL_EINVAL, "this model needs nfields = 2");
  if (p->model == PYCOOL_OSCILLON && nf != 1) return lfail(nullptr, PYCOOL_EINVAL, "oscillon needs nfields = 1");
  if (!(p->mpl > 0)) return lfail(nullptr, PYCOOL_EINVAL, "mpl must be > 0 (+INF = static background)");
  if (p->model == PYCOOL_QBALL && !(p->p[2] > 0)) return lfail(nullptr, PYCOOL_EINVAL, "Q-ball needs M^2 > 0");
  const double* cs = p->stencil;
  const bool dflt = cs[0] == 0 && cs[1] == 0 && cs[2] == 0 && cs[3] == 0;
  if (!dflt) {
    const double s = 6 * cs[1] + 12 * cs[2] + 8 * cs[3];
    if (!(std::fabs(cs[0] + s) <= 1e-12 * (std::fabs(cs[0]) + std::fabs(s))))
      return lfail(nullptr, PYCOOL_EINVAL, "stencil must satisfy c0 = -(6 c1 + 12 c2 + 8 c3)");
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return lfail(nullptr, PYCOOL_ECUDA, "no CUDA device: libpycool has no CPU path");
  }
  pycool_linear_ctx* c = new (std::nothrow) pycool_linear_ctx();
  if (!c) return lfail(nullptr, PYCOOL_ENOMEM, "host allocation failed");
  cudaGetDevice(&c->device);
  cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, c->device);
  c->N = N; c->nf = nf; c->order = order; c->nstages = ns; c->L = L; c->dt = dt;
  for (int i = 0; i < ns; ++i) c->w[i] = w[i];
  c->V = (size_t)N * N * N;
  c->nmodes = (size_t)N * N * (N / 2 + 1);
  c->nclasses = (unsigned)pycool_linear_num_classes(N);
  LinConst& k = c->k;
  k.model = p->model; k.nf = nf;
  for (int i = 0; i < 8; ++i) k.p[i] = p->p[i];
  k.inv_mpl2 = std::isinf(p->mpl) ? 0.0 : 1.0 / (p->mpl * p->mpl);
  k.VL = (double)c->V;
  k.den = 6.0 * k.VL * p->mpl * p->mpl;
  k.rho_g = p->rho_gamma0; k.rho_m = p->rho_m0; k.mpl = p->mpl;
  k.dx2 = (L / N) * (L / N);
  if (dflt) { k.c[0] = -128.0 / 30.0; k.c[1] = 14.0 / 30.0; k.c[2] = 3.0 / 30.0; k.c[3] = 1.0 / 30.0; }   // reading G1
  else for (int i = 0; i < 4; ++i) k.c[i] = cs[i];
  for (int i = 0; i < 4; ++i) c->sc.c[i] = k.c[i];

  const size_t arr = (size_t)nf * c->nmodes * sizeof(double2);
  const size_t mb = (size_t)c->nclasses * 4 * nf * nf * sizeof(double);
  LinBackground b0;
  std::memset(&b0, 0, sizeof b0);
  b0.a = 1.0;
  bool ok = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) == cudaSuccess &&
            cudaMalloc(&c->bg, sizeof(LinBackground)) == cudaSuccess && cudaMalloc(&c->en, sizeof(LinEnergyOut)) == cudaSuccess &&
            cudaMalloc(&c->d_w, 16 * sizeof(double)) == cudaSuccess && cudaMalloc(&c->dPhi, arr) == cudaSuccess &&
            cudaMalloc(&c->dPi, arr) == cudaSuccess && cudaMalloc(&c->M, mb) == cudaSuccess;
  for (int i = 0; ok && i < 4; ++i) ok = cudaEventCreate(&c->ev[i]) == cudaSuccess;
  ok = ok && cudaMemcpyAsync(c->bg, &b0, sizeof b0, cudaMemcpyHostToDevice, c->stream) == cudaSuccess &&
       cudaMemcpyAsync(c->d_w, c->w, 16 * sizeof(double), cudaMemcpyHostToDevice, c->stream) == cudaSuccess &&
       cudaMemsetAsync(c->dPhi, 0, arr, c->stream) == cudaSuccess && cudaMemsetAsync(c->dPi, 0, arr, c->stream) == cudaSuccess &&
       cudaStreamSynchronize(c->stream) == cudaSuccess;
  if (!ok) {
    const cudaError_t e = cudaGetLastError();
    destroy(c);
    return lfail(nullptr, e == cudaErrorMemoryAllocation ? PYCOOL_ENOMEM : PYCOOL_ECUDA,
                 "device set-up failed (%zu bytes of modes, %zu of growth matrices): %s", 2 * arr, mb, cudaGetErrorString(e));
  }
  *out = c;
  return PYCOOL_OK;
}

int pycool_linear_set_background(pycool_linear_ctx* c, double a, double p_a, const double* phi0, const double* pi0) {
  if (!c) return PYCOOL_EINVAL;
  OnDev on(c);
  if (!(a > 0) || !std::isfinite(a)) return lfail(c, PYCOOL_EINVAL, "a must be finite and > 0");
  if (!phi0 || !pi0) return lfail(c, PYCOOL_EINVAL, "phi0 / pi0 is NULL");
  const bool solve = std::isnan(p_a);
  if (solve && std::isinf(c->k.mpl)) return lfail(c, PYCOOL_EINVAL, "p_a = NaN with a static background (mpl = INF)");
  LinBackground b;
  std::memset(&b, 0, sizeof b);
  LIN_TRY(c, cudaMemcpyAsync(&b, c->bg, sizeof b, cudaMemcpyDeviceToHost, c->stream));
  LIN_TRY(c, cudaStreamSynchronize(c->stream));
  b.a = a; b.p_a = solve ? 0.0 : p_a;
  for (int f = 0; f < c->nf; ++f) {
    if (!std::isfinite(phi0[f]) || !std::isfinite(pi0[f])) return lfail(c, PYCOOL_EINVAL, "phi0 / pi0 must be finite");
    b.phi0[f] = phi0[f]; b.pi0[f] = pi0[f];
  }
  LIN_TRY(c, cudaMemcpyAsync(c->bg, &b, sizeof b, cudaMemcpyHostToDevice, c->stream));
  if (solve) {
    lin_set_pa<<<1, 1, 0, c->stream>>>(c->bg, c->k);
    LIN_TRY(c, cudaGetLastError());
  }
  LIN_TRY(c, cudaStreamSynchronize(c->stream));               // b is a stack object
  return PYCOOL_OK;
}

int pycool_linear_set_modes(pycool_linear_ctx* c, const double* dPhi, const double* dPi) {
  if (!c) return PYCOOL_EINVAL;
  OnDev on(c);
  if (!dPhi || !dPi) return lfail(c, PYCOOL_EINVAL, "dPhi_host / dPi_host is NULL");
  const size_t arr = (size_t)c->nf * c->nmodes * sizeof(double2);
  LIN_TRY(c, cudaMemcpyAsync(c->dPhi, dPhi, arr, cudaMemcpyHostToDevice, c->stream));
  LIN_TRY(c, cudaMemcpyAsync(c->dPi, dPi, arr, cudaMemcpyHostToDevice, c->stream));
  lin_zero_mode<<<1, 32, 0, c->stream>>>(c->dPhi, c->dPi, c->nf, c->nmodes);
  LIN_TRY(c, cudaGetLastError());
  LIN_TRY(c, cudaStreamSynchronize(c->stream));
  return PYCOOL_OK;
}

int pycool_linear_set_perturbations(pycool_linear_ctx* c, const double* dphi, const double* dpi) {
  if (!c) return PYCOOL_EINVAL;
  OnDev on(c);
  if (!dphi || !dpi) return lfail(c, PYCOOL_EINVAL, "dphi_host / dpi_host is NULL");
  const CufftApi& fft = cufft_api();
  if (!fft.ok) return lfail(c, PYCOOL_ECUDA, "cuFFT (libcufft.so.11) could not be loaded");
  const int N = c->N;
  double* real = nullptr;
  if (cudaMalloc(&real, c->V * sizeof(double)) != cudaSuccess) {
    cudaGetLastError();
    return lfail(c, PYCOOL_ENOMEM, "out of device memory for the transform scratch");
  }
  cufftHandle plan = 0;
  if (fft.plan3d(&plan, N, N, N, CUFFT_D2Z) != CUFFT_SUCCESS || fft.set_stream(plan, c->stream) != CUFFT_SUCCESS) {
    cudaFree(real);
    return lfail(c, PYCOOL_ENOMEM, "cufftPlan3d(%d^3, D2Z) failed", N);
  }
  int st = PYCOOL_OK;
  for (int which = 0; which < 2 && st == PYCOOL_OK; ++which)
    for (int f = 0; f < c->nf && st == PYCOOL_OK; ++f) {
      const double* src = (which ? dpi : dphi) + (size_t)f * c->V;
      double2* dst = (which ? c->dPi : c->dPhi) + (size_t)f * c->nmodes;
      if (cudaMemcpyAsync(real, src, c->V * sizeof(double), cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
        st = lfail(c, PYCOOL_ECUDA, "H2D copy failed: %s", cudaGetErrorString(cudaGetLastError()));
      else if (fft.exec_d2z(plan, real, (cufftDoubleComplex*)dst) != CUFFT_SUCCESS)
        st = lfail(c, PYCOOL_ECUDA, "cufftExecD2Z failed");
    }
  if (st == PYCOOL_OK) {
    lin_zero_mode<<<1, 32, 0, c->stream>>>(c->dPhi, c->dPi, c->nf, c->nmodes);
    if (cudaGetLastError() != cudaSuccess) st = lfail(c, PYCOOL_ECUDA, "lin_zero_mode launch failed");
  }
  const cudaError_t e = cudaStreamSynchronize(c->stream);
  fft.destroy(plan);
  cudaFree(real);
  if (st != PYCOOL_OK) return st;
  LIN_TRY(c, e);
  return PYCOOL_OK;
}

int pycool_linear_step(pycool_linear_ctx* c, int nsteps, int method) {
  if (!c) return PYCOOL_EINVAL;
  OnDev on(c);
  if (nsteps < 0) return lfail(c, PYCOOL_EINVAL, "nsteps < 0");
  if (method != PYCOOL_LINEAR_GROWTH && method != PYCOOL_LINEAR_NAIVE) return lfail(c, PYCOOL_EINVAL, "unknown method");
  if (nsteps == 0) return PYCOOL_OK;
  switch (c->nf) {
    case 1: return step_t<1>(c, nsteps, method);
    case 2: return step_t<2>(c, nsteps, method);
    case 3: return step_t<3>(c, nsteps, method);
    default: return step_t<4>(c, nsteps, method);
  }
}

int pycool_linear_read_modes(pycool_linear_ctx* c, double* dPhi, double* dPi) {
  if (!c) return PYCOOL_EINVAL;
  OnDev on(c);
  const size_t arr = (size_t)c->nf * c->nmodes * sizeof(double2);
  if (dPhi) LIN_TRY(c, cudaMemcpyAsync(dPhi, c->dPhi, arr, cudaMemcpyDeviceToHost, c->stream));
  if (dPi) LIN_TRY(c, cudaMemcpyAsync(dPi, c->dPi, arr, cudaMemcpyDeviceToHost, c->stream));
  LIN_TRY(c, cudaStreamSynchronize(c->stream));
  return PYCOOL_OK;
}

int pycool_linear_read_perturbations(pycool_linear_ctx* c, double* dphi, double* dpi) {
  if (!c) return PYCOOL_EINVAL;
  OnDev on(c);
  const CufftApi& fft = cufft_api();
  if (!fft.ok) return lfail(c, PYCOOL_ECUDA, "cuFFT (libcufft.so.11) could not be loaded");
  const int N = c->N;
  double2* spec = nullptr;              // Z2D overwrites its input: transform a copy, in place
  if (cudaMalloc(&spec, c->nmodes * sizeof(double2)) != cudaSuccess) {
    cudaGetLastError();
    return lfail(c, PYCOOL_ENOMEM, "out of device memory for the transform scratch");
  }
  cufftHandle plan = 0;
  if (fft.plan3d(&plan, N, N, N, CUFFT_Z2D) != CUFFT_SUCCESS || fft.set_stream(plan, c->stream) != CUFFT_SUCCESS) {
    cudaFree(spec);
    return lfail(c, PYCOOL_ENOMEM, "cufftPlan3d(%d^3, Z2D) failed", N);
  }
  int st = PYCOOL_OK;
  const int nb = (int)std::min<size_t>((c->V + 255) / 256, (size_t)c->sms * 32);
  for (int which = 0; which < 2 && st == PYCOOL_OK; ++which) {
    double* dst = which ? dpi : dphi;
    if (!dst) continue;
    for (int f = 0; f < c->nf && st == PYCOOL_OK; ++f) {
      const double2* src = (which ? c->dPi : c->dPhi) + (size_t)f * c->nmodes;
      if (cudaMemcpyAsync(spec, src, c->nmodes * sizeof(double2), cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess ||
          fft.exec_z2d(plan, (cufftDoubleComplex*)spec, (cufftDoubleReal*)spec) != CUFFT_SUCCESS) {
        st = lfail(c, PYCOOL_ECUDA, "inverse transform failed");
        break;
      }
      // in-place Z2D output rows are padded to 2 (N/2 + 1) doubles
      lin_scale<<<nb, 256, 0, c->stream>>>((double*)spec, 2 * c->nmodes, 1.0 / (double)c->V);
      if (cudaMemcpy2DAsync(dst + (size_t)f * c->V, (size_t)N * sizeof(double), spec, (size_t)(N / 2 + 1) * sizeof(double2),
                            (size_t)N * sizeof(double), (size_t)N * N, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
        st = lfail(c, PYCOOL_ECUDA, "D2H copy failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
  }
  const cudaError_t e = cudaStreamSynchronize(c->stream);
  fft.destroy(plan);
  cudaFree(spec);
  if (st != PYCOOL_OK) return st;
  LIN_TRY(c, e);
  return PYCOOL_OK;
}

int pycool_linear_background_state(pycool_linear_ctx* c, pycool_linear_background* out) {
  if (!c) return PYCOOL_EINVAL;
  OnDev on(c);
  if (!out) return lfail(c, PYCOOL_EINVAL, "out is NULL");
  lin_background_energy<<<1, 1, 0, c->stream>>>(c->bg, c->k, c->en);
  LIN_TRY(c, cudaGetLastError());
  LinBackground b;
  LinEnergyOut e;
  LIN_TRY(c, cudaMemcpyAsync(&b, c->bg, sizeof b, cudaMemcpyDeviceToHost, c->stream));
  LIN_TRY(c, cudaMemcpyAsync(&e, c->en, sizeof e, cudaMemcpyDeviceToHost, c->stream));
  LIN_TRY(c, cudaStreamSynchronize(c->stream));
  std::memset(out, 0, sizeof *out);
  out->a = b.a; out->p_a = b.p_a; out->eta = b.eta;
  for (int f = 0; f < c->nf; ++f) { out->phi0[f] = b.phi0[f]; out->pi0[f] = b.pi0[f]; }
  out->kin = e.kin; out->pot = e.pot; out->rho = e.rho; out->hubble = e.hubble; out->residual = e.residual;
  if (!std::isfinite(b.a) || !std::isfinite(b.p_a)) return lfail(c, PYCOOL_ENONFINITE, "the background became non-finite");
  return PYCOOL_OK;
}

int pycool_linear_growth(pycool_linear_ctx* c, double* M_host, size_t max_classes, size_t* nclasses) {
  if (!c) return PYCOOL_EINVAL;
  OnDev on(c);
  if (nclasses) *nclasses = c->nclasses;
  if (!c->have_growth) return lfail(c, PYCOOL_ESTATE, "no growth matrices yet: call pycool_linear_step(.., PYCOOL_LINEAR_GROWTH)");
  if (!M_host || max_classes < c->nclasses) return lfail(c, PYCOOL_EINVAL, "M_host must hold %u classes", c->nclasses);
  LIN_TRY(c, cudaMemcpyAsync(M_host, c->M, (size_t)c->nclasses * 4 * c->nf * c->nf * sizeof(double), cudaMemcpyDeviceToHost,
                             c->stream));
  LIN_TRY(c, cudaStreamSynchronize(c->stream));
  return PYCOOL_OK;
}

int pycool_linear_time_ms(pycool_linear_ctx* c, double ms[3]) {
  if (!c) return PYCOOL_EINVAL;
  OnDev on(c);
  if (!ms) return lfail(c, PYCOOL_EINVAL, "ms is NULL");
  if (c->last_method < 0) return lfail(c, PYCOOL_ESTATE, "no step yet");
  LIN_TRY(c, cudaStreamSynchronize(c->stream));
  for (int i = 0; i < 3; ++i) {
    float t = 0;
    LIN_TRY(c, cudaEventElapsedTime(&t, c->ev[i], c->ev[i + 1]));
    ms[i] = t;
  }
  if (c->last_method == PYCOOL_LINEAR_NAIVE) ms[1] = 0.0;      // nothing between those two events
  return PYCOOL_OK;
}

int pycool_linear_destroy(pycool_linear_ctx* c) {
  if (!c) return PYCOOL_EINVAL;
  OnDev on(c);
  destroy(c);
  return PYCOOL_OK;
}

const char* pycool_linear_last_error(const pycool_linear_ctx* c) { return c ? c->err.c_str() : g_lin_create_err.c_str(); }

}  // extern "C"

// =============================================================================== growth matrices, no allocation
// pycool_linear_growth_static (include/pycool_linear.h): the growth matrices of (2.51) for callers that cannot
// allocate.  Same kernels as step_t above -- lin_background, lin_growth -- with their scratch (background state, stage
// weights, per-stage coefficient table) in ONE file-scope device array instead of cudaMalloc'ed memory.  Nothing in
// this section allocates: no cudaMalloc / cudaFree, no stream, event or plan creation.
//
// The array's name is a host-side stand-in in host code, not a device address: the host asks for the address once per
// device with cudaGetSymbolAddress (that device current) and passes that pointer to the kernels.  Device code
// (lin_static_seed below) names the array directly.
namespace {

constexpr size_t kMaxStages = PYCOOL_LINEAR_STATIC_MAX_STAGES;
constexpr size_t kStageDoubles = 2 + kLinMaxNF * kLinMaxNF;            // LinStage<4>, the widest

struct StaticScratch {
  LinBackground bg;                          // in/out of lin_background
  double w[16];                              // stage weights
  alignas(256) double table[kMaxStages * kStageDoubles];   // LinStage<NF>[nsteps x nstages], NF <= 4
};
static_assert(sizeof(LinStage<kLinMaxNF>) == kStageDoubles * sizeof(double), "stage layout");
static_assert(sizeof(StaticScratch) == 256 + kMaxStages * kStageDoubles * sizeof(double), "the size pycool_linear.h states");

// 576 KiB + 256 bytes in the device image of every GPU that loads the library.  Shared by every call: see the header.
static __device__ __align__(256) unsigned char g_static_scratch[sizeof(StaticScratch)];

struct SeedArgs {
  LinBackground bg;
  double w[16];
};
// The call's inputs into the scratch, by value through the kernel arguments (no host-to-device copy to wait for).
__global__ void lin_static_seed(const SeedArgs s) {
  StaticScratch* sc = reinterpret_cast<StaticScratch*>(g_static_scratch);
  if (threadIdx.x == 0) sc->bg = s.bg;
  if (threadIdx.x < 16) sc->w[threadIdx.x] = s.w[threadIdx.x];
}

constexpr int kMaxDevices = 64;
std::mutex g_mu;
StaticScratch* g_dev_scratch[kMaxDevices];   // device address of g_static_scratch on device d; nullptr = not asked yet

thread_local std::string g_err = "no error";

int sfail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}
#define ST_TRY(expr)                                                                          \
  do {                                                                                        \
    cudaError_t e_ = (expr);                                                                  \
    if (e_ != cudaSuccess) return sfail(PYCOOL_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

// Once per device, with that device current.
int scratch_of_current_device(StaticScratch** out) {
  int dev = -1;
  ST_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return sfail(PYCOOL_EINVAL, "device ordinal %d is beyond the %d this entry point tracks", dev, kMaxDevices);
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_dev_scratch[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return sfail(PYCOOL_ECUDA, "cudaGetSymbolAddress(static scratch) on device %d: %s", dev, cudaGetErrorString(e));
    }
    g_dev_scratch[dev] = static_cast<StaticScratch*>(p);
  }
  *out = g_dev_scratch[dev];
  return PYCOOL_OK;
}

template <int NF>
int launch(StaticScratch* sc, const SeedArgs& seed, bool solve_pa, const LinConst& k, const LinStencil& st, int N,
           unsigned nclasses, int nstages, int nsteps, double dt, double* M, cudaStream_t stream) {
  LinStage<NF>* table = reinterpret_cast<LinStage<NF>*>(sc->table);
  const size_t nst = (size_t)nsteps * nstages;
  lin_static_seed<<<1, 32, 0, stream>>>(seed);
  ST_TRY(cudaGetLastError());
  if (solve_pa) {
    lin_set_pa<<<1, 1, 0, stream>>>(&sc->bg, k);
    ST_TRY(cudaGetLastError());
  }
  lin_background<NF><<<1, 1, 0, stream>>>(&sc->bg, k, sc->w, nstages, nsteps, dt, table);
  ST_TRY(cudaGetLastError());
  const unsigned long long nthreads = (unsigned long long)nclasses * 2 * NF;
  lin_growth<NF><<<(unsigned)((nthreads + kLinThreads - 1) / kLinThreads), kLinThreads, 0, stream>>>(table, nst, st, N,
                                                                                                     nclasses, M);
  ST_TRY(cudaGetLastError());
  return PYCOOL_OK;
}

}  // namespace

extern "C" {

int pycool_linear_growth_static(int N, double L, int nf, const pycool_params* p, int order, double dt, int nsteps,
                                double a, double p_a, const double* phi0, const double* pi0, double* M_device,
                                size_t max_classes, void* stream) {
  // ---- the checks of pycool_linear_create and pycool_linear_set_background
  if (!p) return sfail(PYCOOL_EINVAL, "params is NULL");
  if (N < 3 || N > 2048 || nf < 1 || nf > kLinMaxNF) return sfail(PYCOOL_EINVAL, "N must be 3..2048, nfields 1..4");
  if (p->precision != 0 && p->precision != 64) return sfail(PYCOOL_EINVAL, "the linearised solver is double precision only");
  if (!(L > 0) || !std::isfinite(L)) return sfail(PYCOOL_EINVAL, "L must be finite and > 0");
  SeedArgs seed;
  std::memset(&seed, 0, sizeof seed);
  const int ns = pycool_stage_weights(order, seed.w, 16);                        // (2.42)-(2.45), Table 1
  if (ns == 0) return sfail(PYCOOL_EINVAL, "order must be 2, 4, 6 or 8");
  if (dt == 0 || !std::isfinite(dt)) return sfail(PYCOOL_EINVAL, "dt must be finite and non-zero");
  if (p->model < PYCOOL_FREE || p->model > PYCOOL_QBALL) return sfail(PYCOOL_EINVAL, "unknown model");
  if ((p->model == PYCOOL_CHAOTIC || p->model == PYCOOL_QBALL) && nf != 2) return sfail(PYCOOL_EINVAL, "this model needs nfields = 2");
  if (p->model == PYCOOL_OSCILLON && nf != 1) return sfail(PYCOOL_EINVAL, "oscillon needs nfields = 1");
  if (!(p->mpl > 0)) return sfail(PYCOOL_EINVAL, "mpl must be > 0 (+INF = static background)");
  if (p->model == PYCOOL_QBALL && !(p->p[2] > 0)) return sfail(PYCOOL_EINVAL, "Q-ball needs M^2 > 0");
  const double* cs = p->stencil;
  const bool dflt = cs[0] == 0 && cs[1] == 0 && cs[2] == 0 && cs[3] == 0;
  if (!dflt) {
    const double s = 6 * cs[1] + 12 * cs[2] + 8 * cs[3];
    if (!(std::fabs(cs[0] + s) <= 1e-12 * (std::fabs(cs[0]) + std::fabs(s))))
      return sfail(PYCOOL_EINVAL, "stencil must satisfy c0 = -(6 c1 + 12 c2 + 8 c3)");
  }
  if (nsteps < 1) return sfail(PYCOOL_EINVAL, "nsteps must be >= 1");
  if ((size_t)nsteps * (size_t)ns > kMaxStages)
    return sfail(PYCOOL_EINVAL, "%d steps x %d stages (order %d) = %zu stages exceed PYCOOL_LINEAR_STATIC_MAX_STAGES = %zu, "
                 "the size of the static scratch: split the call or use pycool_linear_step", nsteps, ns, order,
                 (size_t)nsteps * ns, kMaxStages);
  if (!(a > 0) || !std::isfinite(a)) return sfail(PYCOOL_EINVAL, "a must be finite and > 0");
  if (!phi0 || !pi0) return sfail(PYCOOL_EINVAL, "phi0 / pi0 is NULL");
  const bool solve = std::isnan(p_a);
  if (solve && std::isinf(p->mpl)) return sfail(PYCOOL_EINVAL, "p_a = NaN with a static background (mpl = INF)");
  if (!solve && !std::isfinite(p_a)) return sfail(PYCOOL_EINVAL, "p_a must be finite (or NaN: solve (2.18))");
  seed.bg.a = a; seed.bg.p_a = solve ? 0.0 : p_a;
  for (int f = 0; f < nf; ++f) {
    if (!std::isfinite(phi0[f]) || !std::isfinite(pi0[f])) return sfail(PYCOOL_EINVAL, "phi0 / pi0 must be finite");
    seed.bg.phi0[f] = phi0[f]; seed.bg.pi0[f] = pi0[f];
  }
  const size_t nclasses = pycool_linear_num_classes(N);
  if (!M_device || max_classes < nclasses) return sfail(PYCOOL_EINVAL, "M_device must hold %zu classes", nclasses);

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return sfail(PYCOOL_ECUDA, "no CUDA device: libpycool has no CPU path");
  }
  int dev = -1;
  ST_TRY(cudaGetDevice(&dev));
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, M_device) != cudaSuccess ||
      (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) ||
      (at.type == cudaMemoryTypeDevice && at.device != dev)) {
    cudaGetLastError();
    return sfail(PYCOOL_EINVAL, "M_device is not device memory of the current device (%d)", dev);
  }
  StaticScratch* sc = nullptr;
  if (int st = scratch_of_current_device(&sc)) return st;

  LinConst k;
  std::memset(&k, 0, sizeof k);
  k.model = p->model; k.nf = nf;
  for (int i = 0; i < 8; ++i) k.p[i] = p->p[i];
  k.inv_mpl2 = std::isinf(p->mpl) ? 0.0 : 1.0 / (p->mpl * p->mpl);
  k.VL = (double)((size_t)N * N * N);
  k.den = 6.0 * k.VL * p->mpl * p->mpl;
  k.rho_g = p->rho_gamma0; k.rho_m = p->rho_m0; k.mpl = p->mpl;
  k.dx2 = (L / N) * (L / N);
  if (dflt) { k.c[0] = -128.0 / 30.0; k.c[1] = 14.0 / 30.0; k.c[2] = 3.0 / 30.0; k.c[3] = 1.0 / 30.0; }   // reading G1
  else for (int i = 0; i < 4; ++i) k.c[i] = cs[i];
  LinStencil sten;
  for (int i = 0; i < 4; ++i) sten.c[i] = k.c[i];

  cudaStream_t s = static_cast<cudaStream_t>(stream);
  switch (nf) {
    case 1: return launch<1>(sc, seed, solve, k, sten, N, (unsigned)nclasses, ns, nsteps, dt, M_device, s);
    case 2: return launch<2>(sc, seed, solve, k, sten, N, (unsigned)nclasses, ns, nsteps, dt, M_device, s);
    case 3: return launch<3>(sc, seed, solve, k, sten, N, (unsigned)nclasses, ns, nsteps, dt, M_device, s);
    default: return launch<4>(sc, seed, solve, k, sten, N, (unsigned)nclasses, ns, nsteps, dt, M_device, s);
  }
}

const char* pycool_linear_static_last_error(void) { return g_err.c_str(); }

}  // extern "C"
