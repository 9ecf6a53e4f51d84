/*
 * oracle.h -- C ABI of the CPU oracle for the PyCOOL symplectic step (arXiv 1201.5029 §2.1-2.4).
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_1201_5029_b200/, include/) may
 * include, link or call this.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs use it.  It shares no code with the CUDA path: the struct layouts below are
 * re-declared here on purpose (same field order as include/pycool.h so one ctypes Structure in the
 * harness can describe both, but no common header).
 *
 * What it computes: see the header comment of oracle.cpp (each function cites the passage of
 * PAPER.md it follows).  Single thread, plain loops, no blocking/fusion/reordering.
 */
#ifndef PYCOOL_ORACLE_H
#define PYCOOL_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_ctx oracle_ctx; /* opaque, owned by the library */

enum { ORACLE_OK = 0, ORACLE_EINVAL = 1, ORACLE_ENOMEM = 2, ORACLE_ESTATE = 4, ORACLE_ENONFINITE = 5 };
enum { ORACLE_FREE = 0, ORACLE_CHAOTIC = 1, ORACLE_OSCILLON = 2, ORACLE_QBALL = 3 };

typedef struct {
  int model;          /* enum above */
  double p[8];        /* FREE: m_f^2 per field; CHAOTIC: m^2, g^2; OSCILLON: m^2, lambda, g6;
                         QBALL: m^2, K, M^2, lambda6 */
  double mpl;         /* reduced Planck mass in program units; +INF => static background */
  double rho_gamma0;  /* homogeneous radiation of (2.20) */
  double rho_m0;      /* homogeneous matter of (2.20) */
  double stencil[4];  /* c0..c3 of (2.7); all zero => (-128,14,3,1)/30 */
  int precision;      /* 64 (default when 0), 32, or 80 (long double state; buffers stay double) */
} oracle_params;

typedef struct {
  double a, p_a, eta;
  double kin[4];          /* K_f  = sum pi_f^2 / (2 a^6 V_L)           (2.16) first term  */
  double grad[4];         /* Gr_f = sum G[phi_f] / (2 a^2 dx^2 V_L)    (2.8), (2.16)      */
  double pot;             /* <V>                                                          */
  double rho, pressure;   /* (2.16) + homogeneous components of (2.20)                    */
  double hubble;          /* H = a'/a^2, a' = -p_a/(6 V_L mpl^2)       (2.14)             */
  double residual;        /* |rho/(3 mpl^2 H^2) - 1|                   (3.1)              */
  double sum_phiDphi[4];  /* -sum phi_f D[phi_f] / (2 a^2 dx^2 V_L): equals grad[f] by (2.17) */
} oracle_energy;

/* N: sites per side (>=3); L: box side; order in {2,4,6,8}; dt: conformal step (non-zero). */
int oracle_create(oracle_ctx** out, int N, double L, int nfields, const oracle_params* mp, int order,
                  double dt);
/* phi, pi: nf*N^3 elements each, layout [field][z][y][x], x fastest; element type float if
 * precision==32 else double.  Copied. */
int oracle_set_fields(oracle_ctx*, const void* phi, const void* pi);
/* p_a = NaN => solve the first Friedmann equation (2.18) on the current lattice (expanding branch). */
int oracle_set_background(oracle_ctx*, double a, double p_a);
int oracle_set_dt(oracle_ctx*, double dt);
/* on: dt is a constant PHYSICAL-time increment; step n has conformal length dt / a_n, a_n the scale factor at
 * the start of the step ("adaptive conformal step with constant increases in physical time"). */
int oracle_set_adaptive(oracle_ctx*, int on);
int oracle_step(oracle_ctx*, int nsteps);
int oracle_read_fields(oracle_ctx*, void* phi, void* pi);
int oracle_energies(oracle_ctx*, oracle_energy* out);
int oracle_destroy(oracle_ctx*);
const char* oracle_last_error(const oracle_ctx*);

/* Helpers exposed so tests can pin the pieces separately (not part of the product ABI). */
/* stage weights of one step of the given order, (2.43)-(2.45) + Table 1; returns count, 0 if bad */
int oracle_stage_weights(int order, double* w, int cap);
/* D[phi_f] of (2.7), in lattice units (no 1/dx^2), for field f into out[N^3] (always double) */
int oracle_laplacian(oracle_ctx*, int f, double* out);
/* G[phi_f] of (2.8) per site, lattice units, into out[N^3] */
int oracle_gradient_energy(oracle_ctx*, int f, double* out);
/* V and dV/dphi_f at one point of field space: phi[nf] -> *V, dV[nf] */
int oracle_potential(oracle_ctx*, const double* phi, double* V, double* dV);

#ifdef __cplusplus
}
#endif
#endif
