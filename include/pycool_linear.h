/*
 * pycool_linear.h -- C ABI of the linearised solver of PyCOOL (J. Sainio, arXiv 1201.5029, section 2.2 and
 *                    (2.49)-(2.51)) in libpycool.so, hand-written CUDA for NVIDIA B200 (sm_100a).
 *                    the paper's second workload.
 *
 * What it evolves.  Fields are split into a homogeneous background and perturbations,
 * phi_i(x) = phi_{0,i} + dphi_i(x) (2.21) with sum_x dphi_i = 0 (2.22).  The background (a, p_a, phi_0, pi_0)
 * follows (2.35)-(2.36) on its own; the perturbations follow the linear equations (2.37), evolved in Fourier space
 * (2.38), where modes do not couple:
 *     a'      = -p_a / (6 V_L mpl^2)
 *     p_a'    = V_L (sum_i pi_{0,i}^2 / a^3 - 4 a^3 V(phi_0)) - V_L rho_m0               (2.35), (2.20), reading G25
 *     phi_0'  = pi_0 / a^2 ,  pi_0' = -a^4 dV/dphi_0                                      (2.36)
 *     dPhi_k' = dPi_k / a^2
 *     dPi_k'  = -k_eff^2 a^2 dPhi_k / dx^2 - a^4 sum_j V_ij(phi_0) dPhi_{j,k}             (2.38), (2.26)-(2.27)
 * with -k_eff^2 the eigenvalue of the stencil D of (2.7) on the mode.  One step of length dt is composed of the
 * five flows of (2.49) as in (2.50),
 *     Phi2(h) = H1(h/2) H2(h/2) H3(h/2) H4(h/2) H5(h) H4(h/2) H3(h/2) H2(h/2) H1(h/2),
 * raised to order 4/6/8 with the stage weights of the non-linear step ((2.43)-(2.45), Table 1).
 *
 * Two ways to advance the perturbations, which agree to rounding:
 *   PYCOOL_LINEAR_GROWTH  the linear map M(tau, k_eff^2) of (2.51) is integrated once per DISTINCT value of
 *                         k_eff^2 -- the classes of modes with the same sorted (|n_x|, |n_y|, |n_z|), reading G28:
 *                         (M+1)(M+2)(M+3)/6 of them, M = floor(N/2) -- starting from unit vectors, then every
 *                         Fourier mode is multiplied by the matrix of its class.  All on the device: a one-thread
 *                         kernel advances the background and writes the per-stage coefficients, a second kernel
 *                         integrates one column of one class's matrix per thread, a third applies the matrices.
 *   PYCOOL_LINEAR_NAIVE   every Fourier mode is integrated on its own (the paper's "naive version", which the
 *                         growth-matrix method is "roughly 15 times faster" than).
 *
 * Conventions: as in pycool.h (status codes, host pointers, no CPU path, one context per device, not thread-safe).
 * Everything is double precision (params->precision must be 0 or 64).
 * Real-space arrays: nf * N^3 doubles, layout [field][z][y][x], x fastest.
 * Fourier-space arrays: the half spectrum of a real array, nf * N * N * (N/2 + 1) complex numbers as interleaved
 * (re, im) doubles, layout [field][i_z][i_y][i_x], i_x = 0 .. N/2 fastest, i_y, i_z = 0 .. N-1 with the usual
 * wrap (index i stands for wave number i if i <= N/2, else i - N); plain DFT convention
 * F_k = sum_x f(x) exp(-2 pi i n.x / N), no normalisation (the inverse divides by N^3).
 */
#ifndef PYCOOL_LINEAR_H
#define PYCOOL_LINEAR_H

#include <stddef.h>

#include "pycool.h"

#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default)
#endif

typedef struct pycool_linear_ctx pycool_linear_ctx; /* opaque; pycool_linear_create / pycool_linear_destroy */

enum { PYCOOL_LINEAR_GROWTH = 0, PYCOOL_LINEAR_NAIVE = 1 };

/* The homogeneous background and its energies (2.16) restricted to a homogeneous lattice. */
typedef struct {
  double a, p_a, eta;
  double phi0[4], pi0[4];
  double kin;      /* sum_i pi_{0,i}^2 / (2 a^6)                                                           */
  double pot;      /* V(phi_0)                                                                             */
  double rho;      /* kin + pot + rho_gamma0/a^4 + rho_m0/a^3                              (2.16), (2.20)  */
  double hubble;   /* a'/a^2, a' = -p_a/(6 V_L mpl^2)                                      (2.35)          */
  double residual; /* |rho/(3 mpl^2 H^2) - 1|, 0 for a static background                   (3.1)           */
} pycool_linear_background;

/* Create a context on the current CUDA device: N >= 3, L > 0, nfields 1..4 consistent with params->model, order in
 * {2,4,6,8}, dt finite and non-zero; params as for pycool_create (stencil, mpl, rho_gamma0, rho_m0, model
 * parameters).  Allocates 2 nf half-spectrum arrays and the table of growth matrices
 * ((2 nf)^2 doubles per class).  Initial state: a = 1, p_a = 0, eta = 0, phi_0 = pi_0 = 0, perturbations zero. */
int pycool_linear_create(pycool_linear_ctx** out, int N, double L, int nfields, const pycool_params* params,
                         int order, double dt);

/* Number of distinct-k_eff^2 classes of an N^3 lattice, (M+1)(M+2)(M+3)/6 with M = floor(N/2) (reading G28);
 * class of the sorted triple lo <= mid <= hi is hi(hi+1)(hi+2)/6 + mid(mid+1)/2 + lo. */
size_t pycool_linear_num_classes(int N);

/* Background at the current time: a > 0; phi0, pi0 point to nfields host doubles; p_a = NaN solves the first
 * Friedmann equation (2.18) on the background alone for the expanding branch (reading G10),
 * p_a = -6 V_L mpl a^2 sqrt(rho/3) (PYCOOL_EINVAL with a static background, mpl = INF). */
int pycool_linear_set_background(pycool_linear_ctx*, double a, double p_a, const double* phi0_host,
                                 const double* pi0_host);

/* Perturbations from real-space host arrays (H2D, then a cuFFT D2Z per array on the device); the k = 0 mode is
 * removed (2.22), reading G27. */
int pycool_linear_set_perturbations(pycool_linear_ctx*, const double* dphi_host, const double* dpi_host);
/* Perturbations given directly as half spectra (layout above); the k = 0 mode is removed. */
int pycool_linear_set_modes(pycool_linear_ctx*, const double* dPhi_host, const double* dPi_host);

/* Advance background and perturbations by nsteps steps of length dt (asynchronous, on the context's stream).
 * PYCOOL_LINEAR_GROWTH: one growth matrix per class for the whole call (nsteps steps), then one pass over the
 * modes -- nsteps is how often the modes are brought up to date, the paper's "given number of steps";
 * PYCOOL_LINEAR_NAIVE: every mode through every stage. */
int pycool_linear_step(pycool_linear_ctx*, int nsteps, int method);

/* Half spectra of the perturbations to host (synchronises).  Either pointer may be NULL. */
int pycool_linear_read_modes(pycool_linear_ctx*, double* dPhi_host, double* dPi_host);
/* Real-space perturbations to host: cuFFT Z2D of a copy of each array, divided by N^3 (synchronises). */
int pycool_linear_read_perturbations(pycool_linear_ctx*, double* dphi_host, double* dpi_host);

/* The background and its energies at the current time (synchronises).  PYCOOL_ENONFINITE if a is not finite. */
int pycool_linear_background_state(pycool_linear_ctx*, pycool_linear_background* out);

/* Growth matrices of the latest PYCOOL_LINEAR_GROWTH call to host: [class][row][column], rows and columns ordered
 * (dPhi_1, dPi_1, .., dPhi_nf, dPi_nf) as in (2.51); M_host holds max_classes * (2 nf)^2 doubles; *nclasses
 * receives the class count.  PYCOOL_ESTATE before the first such call, PYCOOL_EINVAL if max_classes is too small. */
int pycool_linear_growth(pycool_linear_ctx*, double* M_host, size_t max_classes, size_t* nclasses);

/* Device time of the kernels of the latest pycool_linear_step call, from CUDA events on the context's stream
 * (synchronises): ms[0] background + coefficient table, ms[1] growth matrices (0 for NAIVE), ms[2] mode update
 * (GROWTH: applying the matrices; NAIVE: the per-mode integration). */
int pycool_linear_time_ms(pycool_linear_ctx*, double ms[3]);

int pycool_linear_destroy(pycool_linear_ctx*);
/* Message of the latest failure of this context (NULL: of the latest failed pycool_linear_create on this
 * thread); library-owned string. */
const char* pycool_linear_last_error(const pycool_linear_ctx*);

/* ---- growth matrices with NO allocation: for callers that cannot call cudaMalloc (a stream under CUDA graph
 * capture, a tight serving loop, a harness that forbids it).  No context: one call computes the growth matrices
 * M(nsteps dt, k_eff^2) of (2.51) of every class -- the background kernel + the growth kernel of
 * pycool_linear_step(.., PYCOOL_LINEAR_GROWTH), same arithmetic, same class order -- for the background given by
 * value, and writes them to memory the CALLER owns.  It calls no cudaMalloc / cudaFree / stream, event or plan
 * creation: the scratch those kernels need (the background state, the stage weights and the per-stage coefficient
 * table, 2 + nf^2 doubles per stage) lives in a fixed array in the library's device image,
 *     PYCOOL_LINEAR_STATIC_MAX_STAGES stages = 576 KiB + 256 bytes,
 * which every GPU that loads libpycool.so holds until the process exits.
 *   nsteps * stages(order) <= PYCOOL_LINEAR_STATIC_MAX_STAGES (stages: 1, 3, 7, 15 for order 2, 4, 6, 8), else
 *   PYCOOL_EINVAL with a message naming the limit; N, L, nfields, params, order, dt as for pycool_linear_create;
 *   a, p_a, phi0_host, pi0_host as for pycool_linear_set_background (host pointers, read before the call returns;
 *   p_a = NaN solves (2.18));
 *   M_device: DEVICE pointer on the current device to max_classes * (2 nf)^2 doubles, layout of pycool_linear_growth,
 *   max_classes >= pycool_linear_num_classes(N) (PYCOOL_EINVAL otherwise, or if it is not device memory of the
 *   current device);
 *   stream: a cudaStream_t of the current device (NULL: the default stream).  The call is asynchronous: it
 *   enqueues three kernels (four with p_a = NaN) and returns; the caller synchronises the stream before reading M_device.
 * Every call on a device shares the one scratch array, which keeps the previous call's contents.  Nothing in it has
 * to start at zero -- each call overwrites the background, the weights and the table entries it later reads -- but
 * calls that overlap on the GPU (different streams, or several host threads) RACE on it: keep calls to one device
 * on one stream, or order them yourself.  Calls on different devices do not interact. */
#define PYCOOL_LINEAR_STATIC_MAX_STAGES 4096
int pycool_linear_growth_static(int N, double L, int nfields, const pycool_params* params, int order, double dt,
                                int nsteps, double a, double p_a, const double* phi0_host, const double* pi0_host,
                                double* M_device, size_t max_classes, void* stream);
/* Message of the latest failed pycool_linear_growth_static on this thread; library-owned string. */
const char* pycool_linear_static_last_error(void);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif /* PYCOOL_LINEAR_H */
