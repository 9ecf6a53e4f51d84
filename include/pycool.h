/*
 * pycool.h -- C ABI of libpycool.so: the non-linear symplectic lattice step of PyCOOL
 *             (J. Sainio, arXiv 1201.5029, §2.1-2.4) as hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * What the library evolves (eq. (2.47)): the state (a, p_a, phi_{f,x}, pi_{f,x}) of nf real
 * scalar fields phi_f and their conjugate momenta pi_f = a^2 phi_f' (2.12) on a periodic N^3 lattice of side
 * L (dx = L/N, V_L = N^3), coupled to the scale factor a and its momentum p_a = -6 a' V_L mpl^2 (2.11) of a
 * flat FRW background, in conformal time eta.  One step of length dt is the composition
 *     step = Phi2(w_1 dt) ... Phi2(w_s dt)                          (2.43)-(2.45), Table 1
 *     Phi2(h) = H1(h/2) H2(h/2) H3(h) H2(h/2) H1(h/2)               (2.48)
 *     H1(e): a   -= p_a/(6 V_L mpl^2) e                              (2.47)
 *     H2(e): p_a += (sum_{f,x} pi^2/a^3 - V_L rho_m0) e;  phi_f += pi_f/a^2 e          "drift"
 *     H3(e): p_a += (a sum phi D[phi]/dx^2 - 4 a^3 sum V) e;
 *            pi_f += (a^2 D[phi_f]/dx^2 - a^4 dV/dphi_f) e                             "kick"
 * with D the 27-point periodic Laplacian stencil (2.7) and the lattice-wide sums computed
 * on the device in a fixed order.  Energies follow (2.16)-(2.20), the residual (3.1).
 *
 * Conventions for every entry point
 *   - returns a status (enum below); never throws, aborts or exits; no CPU fallback exists: without a usable
 *     CUDA device pycool_create returns PYCOOL_ECUDA.
 *   - "host" pointers are caller-owned host memory, read or written only during the call;
 *     "device" pointers are caller-owned CUDA device memory that must stay valid for the life of the context.
 *   - field buffers hold nf*N^3 elements in layout [field][z][y][x] (x fastest); element type is double when
 *     params.precision is 64 (or 0), float when it is 32.  Scalars, sums and energies are always double
 *     (reading G16).
 *   - work is enqueued on the context's CUDA stream; calls that return data synchronise that stream first.
 *   - a context is not thread-safe; distinct contexts are independent.
 *   - a context lives on one CUDA device: the device that is current when pycool_create is called, or the device
 *     that owns d_work for pycool_create_ext.  Every later call switches to that device for its own duration and
 *     restores the caller's current device, so contexts on several GPUs can be driven from one thread
 *     ("many simulations simultaneously").
 */
#ifndef PYCOOL_H
#define PYCOOL_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default) /* the library is built with -fvisibility=hidden: only this ABI is exported */
#endif

typedef struct pycool_ctx pycool_ctx; /* opaque; created by pycool_create*, released by pycool_destroy */

enum {
  PYCOOL_OK = 0,
  PYCOOL_EINVAL = 1,     /* bad argument; pycool_last_error says which                                   */
  PYCOOL_ENOMEM = 2,     /* host or device allocation failed                                             */
  PYCOOL_ECUDA = 3,      /* CUDA runtime error (no device, launch failure, ...)                          */
  PYCOOL_ESTATE = 4,     /* call order: e.g. step before set_fields                                      */
  PYCOOL_ENONFINITE = 5  /* a lattice sum became NaN/Inf; sticky until the next set_fields               */
};

/* Potentials V(phi_1..phi_nf); the derivative dV/dphi_f is compiled in per model (C++ template instance),
 * replacing the paper's run-time code generation. */
enum {
  PYCOOL_FREE = 0,     /* V = sum_f 1/2 m_f^2 phi_f^2                 p = {m_1^2, .., m_nf^2}; nf = 1..4      */
  PYCOOL_CHAOTIC = 1,  /* (3.2) PAPER.md:427: 1/2 m^2 phi^2 + 1/2 g^2 phi^2 chi^2   p = {m^2, g^2}; nf = 2   */
  PYCOOL_OSCILLON = 2, /* (3.3) PAPER.md:456: 1/2 m^2 phi^2 - lambda/4 phi^4 + g6/6 phi^6
                                                                      p = {m^2, lambda, g6}; nf = 1           */
  PYCOOL_QBALL = 3     /* (3.4) PAPER.md:481: m^2 r2 (1 + K ln(r2/M^2)) + lambda6 r2^3/mpl^2,
                          r2 = |Phi|^2 = (phi_1^2+phi_2^2)/2 (reading G7); the log term is 0 for r2 < DBL_MIN
                          (G8)                                        p = {m^2, K, M^2, lambda6}; nf = 2      */
};

typedef struct {
  int model;         /* enum above                                                                        */
  double p[8];       /* model parameters, see enum                                                        */
  double mpl;        /* reduced Planck mass in program units; +INF = static background     */
  double rho_gamma0; /* homogeneous radiation density of (2.20); enters rho only      */
  double rho_m0;     /* homogeneous matter density of (2.20); enters rho and p_a'                         */
  double stencil[4]; /* c_0..c_3 of (2.7) by neighbour class (centre, face, edge, corner).  All zero selects
                        (-128, 14, 3, 1)/30 (reading G1: the paper does not print them).  Must satisfy
                        c_0 = -(6 c_1 + 12 c_2 + 8 c_3), else PYCOOL_EINVAL                               */
  int precision;     /* 64 (also 0) or 32: element type of the field arrays                               */
} pycool_params;

/* Lattice averages at the current (time-synchronised) state.  Always double. */
typedef struct {
  double a, p_a, eta;
  double kin[4];         /* K_f  = sum_x pi_f^2 / (2 a^6 V_L)          first term of (2.16)   */
  double grad[4];        /* Gr_f = sum_x G[phi_f] / (2 a^2 dx^2 V_L)   (2.8) PAPER.md:92                     */
  double pot;            /* <V>                                                                              */
  double rho, pressure;  /* (2.16) plus rho_gamma0/a^4 (+ /3 in P) and rho_m0/a^3 of (2.20)                  */
  double hubble;         /* H = a'/a^2 with a' = -p_a/(6 V_L mpl^2)    (2.14) PAPER.md:123                   */
  double residual;       /* |rho/(3 mpl^2 H^2) - 1|                    (3.1) PAPER.md:415-419; 0 if static   */
  double sum_phiDphi[4]; /* -sum_x phi_f D[phi_f] / (2 a^2 dx^2 V_L); equals grad[f] by (2.17) PAPER.md:146  */
} pycool_energy;

/* Create a context that owns its device memory (2 x the state for ping-pong, plus partial sums) and its own
 * stream.  N >= 3 sites per side; L > 0; nfields 1..4 consistent with the model; order in {2,4,6,8}
 * (stages 1/3/7/15: (2.42), triple jump (2.43)-(2.44) with reading G2, Table 1); dt finite and non-zero
 * (negative runs backwards).  Initial state: a = 1, p_a = 0, eta = 0, no fields.  *out is NULL on failure. */
int pycool_create(pycool_ctx** out, int N, double L, int nfields, const pycool_params* params, int order,
                  double dt);

/* Bytes of device work memory pycool_create_ext needs for this lattice (0 if the arguments are invalid):
 * both state buffers in the library's internal layout (ghost columns/rows for even N), partial sums, scalars. */
size_t pycool_work_bytes(int N, int nfields, int precision);

/* As pycool_create, on caller-owned device memory and stream (e.g. a PyTorch tensor / torch stream):
 *   d_work      : device, >= pycool_work_bytes(...) bytes, 256-byte aligned; holds the whole state
 *   cuda_stream : a cudaStream_t (NULL = the legacy default stream)
 * The caller keeps ownership; pycool_destroy frees neither. */
int pycool_create_ext(pycool_ctx** out, int N, double L, int nfields, const pycool_params* params, int order,
                      double dt, void* d_work, size_t work_bytes, void* cuda_stream);

/* Upload phi and pi from dense host arrays [field][z][y][x] (H2D on the context stream, synchronous to the
 * caller), write the periodic ghost images and compute sum pi^2 on the device.  Clears PYCOOL_ENONFINITE. */
int pycool_set_fields(pycool_ctx*, const void* phi_host, const void* pi_host);
/* Same from dense device arrays (D2D on the context stream, asynchronous). */
int pycool_set_fields_device(pycool_ctx*, const void* d_phi_src, const void* d_pi_src);

/* Seeded Gaussian initial conditions generated on the device (the paper takes its
 * fluctuations from Defrost without describing the generator, so the recipe is DESIGN.md's reading
 * G21).  Array (field f, phi or pi) = mean + a real Gaussian random field with spectrum
 *     A(k) = amp (k^2 + m2)^q   for 0 < k <= kmax (kmax <= 0: every k),   k = 2 pi |n| / L,
 * F_k = A(k)(g1 + i g2)/sqrt 2 with (g1, g2) from Philox4x32-10(counter = (mode index, array id 2f | 2f+1), key =
 * seed) through Box-Muller, field = mean + sqrt(2)/L^1.5 sum_k F_k exp(2 pi i n.x/N) (cuFFT, loaded on demand).
 * Vacuum fluctuations |phi_k|^2 = 1/(2 omega_k): amp = c/sqrt 2, q = -1/4 for phi and +1/4 for pi, m2 = m_eff^2.
 * phi_spec, pi_spec: nfields entries each (host).  Replaces set_fields; even N only.  Synchronises.  The same seed
 * gives the same lattice on any GPU.  Scratch: one N^2 (N/2 + 1) x 16-byte buffer plus cuFFT's work area. */
typedef struct { double mean, amp, m2, q, kmax; } pycool_spectrum;
int pycool_init_fields(pycool_ctx*, unsigned long long seed, const pycool_spectrum* phi_spec,
                       const pycool_spectrum* pi_spec);

/* Shell-summed spectrum of one array (the paper's spectra are LATTICEEASY's and Defrost's,
 * not defined in it: this is the field spectrum they are all built from, reading G22).  With
 * F_k = L^1.5 / (sqrt 2 N^3) sum_x field(x) exp(-2 pi i n.x/N) -- the convention of pycool_init_fields turned around,
 * so a field made with spectrum A(k) gives <power/count> = A(k)^2 --
 *   power[i] = sum |F_k|^2 and count[i] = number of modes over the full spectrum with round(|n|) = i, i < nbins
 * (nbins = round(sqrt 3 N/2) + 1 covers every mode; 1 <= nbins <= 3072; the mean sits in power[0]).  field in [0, nfields), which = 0
 * for phi, 1 for pi.  cuFFT D2Z on a double copy; the shell sums use atomics, so the last bits are not
 * reproducible from run to run.  Applies a pending closing drift first.  Synchronises. */
int pycool_field_spectrum(pycool_ctx*, int field, int which, int nbins, double* power_host, double* count_host);

/* Number-density and energy-density spectra of one field (the paper's post-processing writes
 * "field, number density and energy density spectra that are used in LATTICEEASY", and defines none of
 * them: reading G24).  They are the spectra of the DISCRETE Hamiltonian (2.20) that the step integrates: with
 * F^phi_k, F^pi_k as in pycool_field_spectrum, the canonical pair u_k = a F^phi_k, v_k = F^pi_k / a and
 *     w_k^2 = k_eff^2(n) / dx^2 + a^2 m_eff2,   -k_eff^2 = eigenvalue of the stencil (2.7) on the mode,
 *     n_k   = 1/2 (w_k |u_k|^2 + |v_k|^2 / w_k)     (0 where w_k^2 <= 0),      rho_k = 1/2 (|v_k|^2 + w_k^2 |u_k|^2),
 * number[i], energy[i], count[i] = sums over the modes of the full spectrum with round(|n|) = i, i < nbins <= 2048.
 * Then (2 / (a^4 L^3)) sum_i energy[i] = kin[f] + grad[f] + 1/2 m_eff2 <phi_f^2> of pycool_energies exactly
 * (Parseval), and a vacuum state made by pycool_init_fields (|phi_k|^2 = 1/(2 w_k)) has number/count = 1/2.
 * a is the current (time-synchronised) scale factor; m_eff2 is the caller's effective mass squared of the field
 * (e.g. d^2V/dphi^2 at the mean field).  Two cuFFT D2Z transforms; applies a pending closing drift first.
 * Synchronises. */
int pycool_mode_spectra(pycool_ctx*, int field, double m_eff2, int nbins, double* number_host, double* energy_host,
                        double* count_host);

/* Set a (> 0) and p_a.  p_a = NaN asks the library to solve the first Friedmann equation (2.18) on the
 * current lattice, expanding branch (reading G10): p_a = -6 V_L mpl a^2 sqrt(rho/3); needs fields and a
 * finite mpl.  With mpl = +INF pass p_a = 0. */
int pycool_set_background(pycool_ctx*, double a, double p_a);

int pycool_set_dt(pycool_ctx*, double dt);

/* on != 0: dt becomes a constant PHYSICAL-time increment: step n has conformal length dt / a_n, a_n the scale
 * factor at the start of that step, computed on the device ("adaptive conformal step with constant increases in
 * physical time").  pycool_energy.eta is the sum of the lengths.  Default off. */
int pycool_set_adaptive(pycool_ctx*, int on);

/* Advance nsteps >= 0 whole steps of length dt.  Asynchronous: kernels are enqueued on the context stream
 * (no host synchronisation inside, a and p_a live on the device).  On return from a later synchronising call
 * the state is time-synchronised at eta + nsteps*dt.  Returns PYCOOL_ENONFINITE if an EARLIER call left the
 * sticky flag set and it has been observed by a synchronising call. */
int pycool_step(pycool_ctx*, int nsteps);

/* The closing half drift H2(h_s/2) of a pycool_step call ((2.48)) is deferred: a following
 * pycool_step merges it with its own opening half drift exactly as between two stages of one call, so
 * step(1) x n and step(n) give bitwise the same state; every call that looks at the fields (read_fields*,
 * device_fields, energies, set_background, sync) applies it first.  pycool_flush applies it now (asynchronous,
 * one pointwise pass over phi); a no-op when nothing is pending. */
int pycool_flush(pycool_ctx*);

/* Apply a pending closing drift and wait for the context stream; returns PYCOOL_ENONFINITE / PYCOOL_ECUDA if
 * the enqueued work failed. */
int pycool_sync(pycool_ctx*);

/* Download phi and/or pi (either may be NULL) to host memory.  Synchronises. */
int pycool_read_fields(pycool_ctx*, void* phi_host, void* pi_host);

/* Download into dense device arrays (either may be NULL).  D2D on the context stream, asynchronous. */
int pycool_read_fields_device(pycool_ctx*, void* d_phi_dst, void* d_pi_dst);

/* Device pointers of the current state arrays (they alternate between the two state buffers; valid until
 * the next pycool_step/set_fields) and their layout: element (f, z, y, x) is at
 *   ((f*N + z)*layout[1] + y + layout[3]) * layout[0] + x + layout[2]
 * (layout = row pitch, rows per plane, ghost columns, ghost rows).  Does not synchronise. */
int pycool_device_fields(pycool_ctx*, void** d_phi, void** d_pi, size_t layout[4]);

/* Lattice sums of the current state (one stencil pass with G of (2.8)) -> rho, P, H, residual.
 * Synchronises. */
int pycool_energies(pycool_ctx*, pycool_energy* out);

/* Energy log: "How frequently to calculate the energy densities and to write them to a file is decided by the
 * user".  every > 0: after every `every`-th completed step (counted from this call) pycool_step
 * enqueues an energy read-out of the state that step ends in -- the lattice sums seen through the step's closing
 * half drift, at the scale factor of that instant, finished on the device (rho, P, H, residual) -- and appends it
 * to a device ring buffer of `capacity` entries.  No host synchronisation, and the step sequence itself is
 * untouched: fields and scalars are bitwise those of an unlogged run, and every entry is bitwise what
 * pycool_energies returns for a run stopped at that step.  every = 0 switches the log off and frees it.
 * pycool_read_energy_log copies the newest min(logged, capacity, max_entries) entries, oldest first, to host memory
 * (*n_out of them; *total, if not NULL, = entries logged since the cadence was set).  Synchronises. */
int pycool_set_energy_cadence(pycool_ctx*, int every, int capacity);
int pycool_read_energy_log(pycool_ctx*, pycool_energy* out_host, int max_entries, int* n_out,
                           unsigned long long* total);

int pycool_destroy(pycool_ctx*);

/* Library-owned, NUL-terminated description of the last error of this context (valid until the next call
 * on it); a static string for ctx == NULL. */
const char* pycool_last_error(const pycool_ctx*);

/* Stage weights w_1..w_s of one step of the given order into w[cap]; returns s, or 0 if order is not
 * supported or cap < s.  (2.42)-(2.45), Table 1. */
int pycool_stage_weights(int order, double* w, int cap);

/* ---- instrumentation (does not change results) ---- */
/* Number of kernels this context has launched so far, by kind:
 *   counts[0] fused drift+kick (stages: a cooperative multi-stage launch counts each of its stages),
 *   [1] reduce+scalar update, [2] closing drift, [3] energy/sum kernels. */
int pycool_launch_counts(const pycool_ctx*, unsigned long long counts[4]);
/* profiling on: bracket every fused drift+kick launch with CUDA events on the context stream. */
int pycool_set_profiling(pycool_ctx*, int on);
/* Sum of the bracketed durations (ms) and their number since profiling was switched on.  Synchronises. */
int pycool_kick_time_ms(pycool_ctx*, double* total_ms, unsigned long long* launches);
/* Launch geometry of the fused kernel: tile[0..2] = TX, TY, z-chunk; tile[3] = threads per block;
 * tile[4] = work items (x-y tile, z-chunk) per launch -- the grid size of a one-block-per-item launch; a persistent
 * launch uses min(items, resident blocks) blocks; tile[5] = dynamic shared memory bytes; tile[6] = variant index
 * (pycool_set_tile);
 * tile[7] = TMA ring stages (0 = the register-prefetch kernel); tile[8], tile[9] = region of the item order in tiles
 * (x: always the whole row; y: rows per region; pycool_set_item_order; the whole x-y tile grid = plain order). */
int pycool_kick_geometry(const pycool_ctx*, int tile[10]);
/* Override the z-chunk length (planes per block; 0 = automatic) before the next step. */
int pycool_set_zchunk(pycool_ctx*, int planes);
/* Fused stage tail (default on): the block of a drift+kick launch that finishes last adds the per-block partial
 * sums in block-index order and advances a, p_a and the next stage's coefficients,
 * so a stage is ONE launch.  Off: a separate reduce + scalar-update launch follows every kick.  Both orders of
 * summation are fixed; they differ from each other in the last bits only. */
int pycool_set_fused_tail(pycool_ctx*, int on);
/* Small lattices (default on): when every work item of a stage fits on the GPU at once (32^3 .. 128^3 on a B200) and
 * the device supports cooperative launches, pycool_step runs up to 32 steps' worth of stages in ONE cooperative launch,
 * with a grid-wide barrier between stages instead of a kernel boundary (the paper goes back to the CPU at every
 * sub-step).  Results are bitwise those of the launch-per-stage path.  Off, while profiling, with the
 * fused tail off or for larger lattices: one launch per stage.  pycool_launch_counts counts stages either way. */
int pycool_set_cooperative(pycool_ctx*, int on);
/* Programmatic dependent launch of the TMA-fed kernel (default on): the next stage's blocks are scheduled while
 * the current stage drains and wait (griddepcontrol.wait) until it has completed before they read anything it
 * wrote.  Hides launch latency and prologue on small lattices; results are unchanged. */
int pycool_set_overlap(pycool_ctx*, int on);
/* Order in which the persistent TMA-fed kernel hands out its work items (x-y tile, z-chunk).  -1 (default): the x-y
 * tile grid is cut into regions of whole tile rows holding about as many tiles as there are blocks in flight, and a
 * region is taken through ALL its z-chunks before the next region, so the blocks that finish z-chunk k of a region
 * go on with z-chunk k+1 of the same tiles and the two planes consecutive chunks share are read from L2 the second
 * time; 0: plain order (every tile of z-chunk 0, then z-chunk 1, ...); n > 0: regions of about n tiles.
 * Fields do not depend on the order; the lattice sums are added in item-index order, so they change in the last
 * bits with it (each order is reproducible bit for bit). */
int pycool_set_item_order(pycool_ctx*, int tiles_per_region);
/* pycool_energies kernel: 1 (default) = TMA-fed z-march (even N, at most two fields; sum_x G[phi] through the paper's
 * identity (2.17), sum_x G = -sum_x psi D[psi] with psi = phi - one lattice-wide reference value per field);
 * 0 = the plain one-thread-per-site kernel that evaluates (2.8) term by term (always used for odd N or more than two
 * fields).  They agree to rounding.  2, 3, 4 pick the TMA kernel's tile (64x16 with 2x2 sites per thread; 32x16 with
 * 2x1 sites and two blocks per SM; 32x16 with 2x2 sites) instead of the automatic choice. */
int pycool_set_energy_kernel(pycool_ctx*, int tma);
/* Persistent launch of the TMA-fed kernel (default on): as many blocks as fit on the device at once; a block's
 * first work item (x-y tile, z-chunk) is its index, every further one is claimed from a device counter
 * (atomicAdd) in index order -- the order a hardware block scheduler would hand them out, which keeps the blocks
 * in flight x-y neighbours (a static round-robin deal was measured 1.5x slower) -- with the TMA ring
 * running on across item boundaries.  Off: one block per work item.  Partial sums are indexed by work item, so
 * results are bitwise the same whichever block computes what. */
int pycool_set_persistent(pycool_ctx*, int on);
/* Select the variant of the fused kernel; -1 = automatic (by model, precision, number of fields and N).
 *   0..2: register-prefetch kernel, x-y tiles 32x8, 32x16, 64x8 sites (any N);
 *   3..10: TMA-fed kernel (even N >= 4 only, else PYCOOL_EINVAL): tiles 64x16, 32x16, 128x8, 128x16 with 2 x 2
 *         sites per thread; 32x16, 64x8 with 2 x 1 sites per thread and two blocks per SM; 128x16 with 2 x 4
 *         sites per thread (one-field lattices); 32x16 with 2 x 1 sites per thread, one block per SM (three and
 *         four fp64 fields);
 *   11:   128x8 as x quads, 4 x 1 sites per thread with 16-byte float accesses (fp32 only, N a multiple of 4);
 *   12:   32x8 with 2 x 1 sites per thread and four blocks per SM (the Q-ball model in fp64 only).
 * PYCOOL_EINVAL also if the variant's TMA ring does not fit in shared memory for this model and precision, or
 * if its per-thread state would not fit the register budget for this number of fields (such instances are not
 * compiled: no variant that spills is shipped). */
int pycool_set_tile(pycool_ctx*, int tile);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif /* PYCOOL_H */
