/*
 * oracle.cpp -- plain, slow, single-threaded CPU oracle for the PyCOOL non-linear symplectic step.
 *
 * TEST INFRASTRUCTURE ONLY (see oracle.h).  Written from /root/reference/PAPER.md (arXiv 1201.5029);
 * shares no code with the CUDA path.  Compile with -ffp-contract=off (build.py does).
 *
 * The method is an integrator, so the oracle is the algorithm step by step in the paper's order:
 *
 *   state  (a, p_a, phi_{f,x}, pi_{f,x})                                   PAPER.md:325-332 (2.47)
 *   step   = Phi2(w_1 dt) ... Phi2(w_s dt)                                 PAPER.md:293-310 (2.43)-(2.45), Table 1
 *   Phi2(h)= H1(h/2) H2(h/2) H3(h) H2(h/2) H1(h/2)                         PAPER.md:334-336 (2.48)
 *   H1(e): a   -= p_a/(6 V_L mpl^2) e
 *   H2(e): p_a += (sum pi^2 / a^3 - V_L rho_m0) e ; phi += pi/a^2 e
 *   H3(e): p_a += (a sum phi D[phi]/dx^2 - 4 a^3 sum V) e ;
 *          pi  += (a^2 D[phi]/dx^2 - a^4 dV/dphi) e
 *   D[phi] = sum_alpha c_d(alpha) phi(alpha), 27 points, periodic          PAPER.md:85-90 (2.7)
 *   G[phi] = 1/2 sum_alpha c_d (phi(alpha)-phi(x))^2                       PAPER.md:92 (2.8)
 *   rho, P                                                                 PAPER.md:139-144 (2.16), 162 (2.20)
 *   residual |rho/(3 mpl^2 H^2) - 1|                                       PAPER.md:415-419 (3.1)
 *
 * Readings of silent/garbled points:
 *   G1  default weights (c0..c3) = (-128,14,3,1)/30; run-time parameters.
 *   G2  z1 = 1/(2-2^(1/3)), z0 = -2^(1/3)/(2-2^(1/3))  (the printed z0 denominator is garbled).
 *   G7  |Phi|^2 = (phi1^2+phi2^2)/2.   G8 log term := 0 when r^2 < DBL_MIN.
 *   G10 p_a from (2.18) on the expanding branch.   G16 fp32 fields keep fp64 scalars and sums.
 *   D[phi] is evaluated in difference form sum c_d (phi(alpha)-phi(x)), identical to (2.7)
 *   because c0 = -(6c1+12c2+8c3) (checked at create), to avoid cancellation against the
 *   homogeneous part of phi.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): P1-P13 of SURVEY.md 8(c).  Nothing here is
 * "parity unpinned".
 */
#include "oracle.h"

#include <cfloat>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <new>
#include <string>
#include <vector>

namespace {

/* Neumaier-compensated accumulator in long double: the oracle is the accurate side of every sum. */
struct Sum {
  long double s = 0.0L, c = 0.0L;
  void add(long double v) {
    long double t = s + v;
    if (fabsl(s) >= fabsl(v)) c += (s - t) + v; else c += (v - t) + s;
    s = t;
  }
  long double value() const { return s + c; }
};

/* Stage weights: Table 1.  Returns count. */
int stage_weights(int order, long double* w) {
  if (order == 2) { w[0] = 1.0L; return 1; }
  if (order == 4) {                         /* (2.43)-(2.44) with n=1, reading G2 */
    long double c = cbrtl(2.0L);
    long double z1 = 1.0L / (2.0L - c), z0 = -c / (2.0L - c);
    w[0] = z1; w[1] = z0; w[2] = z1; return 3;
  }
  if (order == 6) {                         /* Table 1, 7 stages, w_{s+1-i} = w_i */
    long double w1 = 0.78451361047755726382L, w2 = 0.23557321335935813368L,
                w3 = -1.17767998417887100695L;
    long double w4 = 1.0L - 2.0L * (w1 + w2 + w3);
    long double v[7] = {w1, w2, w3, w4, w3, w2, w1};
    for (int i = 0; i < 7; ++i) w[i] = v[i];
    return 7;
  }
  if (order == 8) {                         /* Table 1, 15 stages */
    long double h[8] = {0.74167036435061295345L, -0.40910082580003159400L, 0.19075471029623837995L,
                        -0.57386247111608226666L, 0.29906418130365592384L, 0.33462491824529818378L,
                        0.31529309239676659663L, 0.0L};
    long double s = 0.0L;
    for (int i = 0; i < 7; ++i) s += h[i];
    h[7] = 1.0L - 2.0L * s;
    for (int i = 0; i < 8; ++i) { w[i] = h[i]; w[14 - i] = h[i]; }
    return 15;
  }
  return 0;
}

struct Base {
  virtual ~Base() {}
  std::string err;
  virtual int set_fields(const void*, const void*) = 0;
  virtual int set_background(double, double) = 0;
  virtual int set_dt(double) = 0;
  virtual int set_adaptive(int) = 0;
  virtual int step(int) = 0;
  virtual int read_fields(void*, void*) = 0;
  virtual int energies(oracle_energy*) = 0;
  virtual int laplacian(int, double*) = 0;
  virtual int gradient_energy(int, double*) = 0;
  virtual int potential(const double*, double*, double*) = 0;
};

/* T = field element type; S = type of a, p_a and the sums' results; IO = buffer element type. */
template <class T, class S, class IO>
struct Stepper : Base {
  int N, nf, order;
  size_t V;             /* V_L = N^3 */
  S L, dx, dt, mpl, rho_g, rho_m;
  S a, p_a, eta;
  int model;
  S par[8];
  S c[4];               /* stencil weights by neighbour class d = 0..3 */
  std::vector<T> phi, pi;
  bool have_fields = false, nonfinite = false;
  bool adaptive = false;  /* dt is a physical-time increment: each step uses d eta = dt / a */

  size_t idx(int f, int x, int y, int z) const {
    return (size_t)f * V + ((size_t)z * N + (size_t)y) * N + (size_t)x;
  }
  int wrap(int i) const { return (i % N + N) % N; }   /* periodic lattice */

  /* ---- potentials: V and dV/dphi_f.  PAPER.md:427 (3.2), 456 (3.3), 481 (3.4) ---- */
  S pot(const S* p, S* dV) const {
    switch (model) {
      case ORACLE_FREE: {                    /* V = sum_f 1/2 m_f^2 phi_f^2 */
        S v = 0;
        for (int f = 0; f < nf; ++f) { v += S(0.5) * par[f] * p[f] * p[f]; dV[f] = par[f] * p[f]; }
        return v;
      }
      case ORACLE_CHAOTIC: {                 /* (3.2): V = 1/2 m^2 phi^2 + 1/2 g^2 phi^2 chi^2 */
        S m2 = par[0], g2 = par[1];
        S ph = p[0], ch = p[1];
        dV[0] = m2 * ph + g2 * ph * ch * ch;
        dV[1] = g2 * ph * ph * ch;
        return S(0.5) * m2 * ph * ph + S(0.5) * g2 * ph * ph * ch * ch;
      }
      case ORACLE_OSCILLON: {                /* (3.3), reading G6: 1/2 m^2 phi^2 - l/4 phi^4 + g6/6 phi^6 */
        S m2 = par[0], lam = par[1], g6 = par[2];
        S ph = p[0], p2 = ph * ph;
        dV[0] = m2 * ph - lam * p2 * ph + g6 * p2 * p2 * ph;
        return S(0.5) * m2 * p2 - lam / S(4) * p2 * p2 + g6 / S(6) * p2 * p2 * p2;
      }
      case ORACLE_QBALL: {                   /* (3.4), readings G6-G8; gH^2 term omitted */
        S m2 = par[0], K = par[1], M2 = par[2], l6 = par[3];
        S r2 = (p[0] * p[0] + p[1] * p[1]) / S(2);
        S lg = (r2 < S(DBL_MIN)) ? S(0) : S(std::log(r2 / M2));
        S six = l6 / (mpl * mpl);            /* 0 when mpl = +INF */
        S common = m2 * (S(1) + K + K * lg) + S(3) * six * r2 * r2;
        dV[0] = common * p[0];
        dV[1] = common * p[1];
        return m2 * r2 * (S(1) + K * lg) + six * r2 * r2 * r2;
      }
    }
    return 0;
  }

  /* ---- D[phi_f](x,y,z), (2.7), difference form, lattice units ---- */
  S lap(int f, int x, int y, int z) const {
    S ctr = S(phi[idx(f, x, y, z)]);
    S s[4] = {0, 0, 0, 0};
    for (int dz = -1; dz <= 1; ++dz)
      for (int dy = -1; dy <= 1; ++dy)
        for (int dxi = -1; dxi <= 1; ++dxi) {
          int d = (dxi != 0) + (dy != 0) + (dz != 0);   /* neighbour class */
          if (d == 0) continue;
          s[d] += S(phi[idx(f, wrap(x + dxi), wrap(y + dy), wrap(z + dz))]) - ctr;
        }
    return c[1] * s[1] + c[2] * s[2] + c[3] * s[3];
  }

  /* ---- G[phi_f](x,y,z), (2.8), lattice units ---- */
  S grad_e(int f, int x, int y, int z) const {
    S ctr = S(phi[idx(f, x, y, z)]);
    S s[4] = {0, 0, 0, 0};
    for (int dz = -1; dz <= 1; ++dz)
      for (int dy = -1; dy <= 1; ++dy)
        for (int dxi = -1; dxi <= 1; ++dxi) {
          int d = (dxi != 0) + (dy != 0) + (dz != 0);
          if (d == 0) continue;
          S df = S(phi[idx(f, wrap(x + dxi), wrap(y + dy), wrap(z + dz))]) - ctr;
          s[d] += df * df;
        }
    return S(0.5) * (c[1] * s[1] + c[2] * s[2] + c[3] * s[3]);
  }

  /* ---- the three exact flows of (2.47) ---- */
  void H1(S e) { a -= p_a / (S(6) * S(V) * mpl * mpl) * e; }

  void H2(S e) {
    Sum sp;
    for (size_t i = 0; i < (size_t)nf * V; ++i) sp.add((long double)pi[i] * (long double)pi[i]);
    S Spi = S(sp.value());
    if (!std::isfinite((double)Spi)) nonfinite = true;
    p_a += (Spi / (a * a * a) - S(V) * rho_m) * e;
    S k = e / (a * a);
    for (size_t i = 0; i < (size_t)nf * V; ++i) phi[i] = T(S(phi[i]) + S(pi[i]) * k);
  }

  void H3(S e) {
    Sum sD, sV;
    S kD = a * a / (dx * dx) * e, kV = a * a * a * a * e;
    S p[4], dV[4], D[4];
    for (int z = 0; z < N; ++z)
      for (int y = 0; y < N; ++y)
        for (int x = 0; x < N; ++x) {
          for (int f = 0; f < nf; ++f) {
            p[f] = S(phi[idx(f, x, y, z)]);
            D[f] = lap(f, x, y, z);
            sD.add((long double)p[f] * (long double)D[f]);
          }
          S v = pot(p, dV);
          sV.add((long double)v);
          /* pi is updated in place: D reads only phi, which H3 leaves unchanged */
          for (int f = 0; f < nf; ++f) {
            size_t i = idx(f, x, y, z);
            pi[i] = T(S(pi[i]) + kD * D[f] - kV * dV[f]);
          }
        }
    S SD = S(sD.value()), SV = S(sV.value());
    if (!std::isfinite((double)SD) || !std::isfinite((double)SV)) nonfinite = true;
    p_a += (a * SD / (dx * dx) - S(4) * a * a * a * SV) * e;
  }

  void phi2(S h) {                                                          /* (2.48) */
    H1(h / S(2));
    H2(h / S(2));
    H3(h);
    H2(h / S(2));
    H1(h / S(2));
  }

  int step(int n) override {
    if (!have_fields) { err = "step before set_fields"; return ORACLE_ESTATE; }
    if (n < 0) { err = "nsteps < 0"; return ORACLE_EINVAL; }
    long double w[16];
    int s = stage_weights(order, w);
    for (int it = 0; it < n; ++it) {
      /* "adaptive conformal step with constant increases in physical time": dt_phys = a d eta,
         so the conformal length of this step is dt / a with a taken at the start of the step (reading G20) */
      const S de = adaptive ? dt / a : dt;
      for (int i = 0; i < s; ++i) phi2(S(w[i]) * de);                       /* (2.43)/(2.45) */
      eta += de;
    }
    if (nonfinite) { err = "non-finite lattice sum"; return ORACLE_ENONFINITE; }
    return ORACLE_OK;
  }

  int set_fields(const void* ph, const void* pp) override {
    if (!ph || !pp) { err = "null buffer"; return ORACLE_EINVAL; }
    const IO* a1 = (const IO*)ph; const IO* a2 = (const IO*)pp;
    for (size_t i = 0; i < (size_t)nf * V; ++i) { phi[i] = T(a1[i]); pi[i] = T(a2[i]); }
    have_fields = true; nonfinite = false;
    return ORACLE_OK;
  }

  int read_fields(void* ph, void* pp) override {
    if (!have_fields) { err = "read before set_fields"; return ORACLE_ESTATE; }
    IO* a1 = (IO*)ph; IO* a2 = (IO*)pp;
    for (size_t i = 0; i < (size_t)nf * V; ++i) {
      if (a1) a1[i] = IO(phi[i]);
      if (a2) a2[i] = IO(pi[i]);
    }
    return ORACLE_OK;
  }

  /* lattice averages that enter rho and P, at scale factor a */
  void averages(S* K, S* Gr, S* GrD, S* Vbar) const {
    S a2 = a * a, a6 = a2 * a2 * a2, Vs = S(V);
    for (int f = 0; f < nf; ++f) {
      Sum sp, sg, sd;
      for (int z = 0; z < N; ++z)
        for (int y = 0; y < N; ++y)
          for (int x = 0; x < N; ++x) {
            size_t i = idx(f, x, y, z);
            sp.add((long double)pi[i] * (long double)pi[i]);
            sg.add((long double)grad_e(f, x, y, z));
            sd.add((long double)S(phi[i]) * (long double)lap(f, x, y, z));
          }
      K[f] = S(sp.value()) / (S(2) * a6 * Vs);                 /* phi'^2/(2a^2), phi' = pi/a^2 (2.12) */
      Gr[f] = S(sg.value()) / (S(2) * a2 * dx * dx * Vs);      /* (grad phi)^2/(2a^2) via (2.8)      */
      GrD[f] = -S(sd.value()) / (S(2) * a2 * dx * dx * Vs);    /* same via (2.17)                    */
    }
    Sum sv;
    S p[4], dV[4];
    for (int z = 0; z < N; ++z)
      for (int y = 0; y < N; ++y)
        for (int x = 0; x < N; ++x) {
          for (int f = 0; f < nf; ++f) p[f] = S(phi[idx(f, x, y, z)]);
          sv.add((long double)pot(p, dV));
        }
    *Vbar = S(sv.value()) / Vs;
  }

  int energies(oracle_energy* o) override {
    if (!o) { err = "null out"; return ORACLE_EINVAL; }
    if (!have_fields) { err = "energies before set_fields"; return ORACLE_ESTATE; }
    S K[4], Gr[4], GrD[4], Vbar;
    averages(K, Gr, GrD, &Vbar);
    std::memset(o, 0, sizeof(*o));
    S a2 = a * a;
    S rho = Vbar + rho_g / (a2 * a2) + rho_m / (a2 * a);                    /* (2.16) + (2.20) */
    S P = -Vbar + rho_g / (S(3) * a2 * a2);
    for (int f = 0; f < nf; ++f) {
      rho += K[f] + Gr[f];
      P += K[f] - Gr[f] / S(3);
      o->kin[f] = (double)K[f]; o->grad[f] = (double)Gr[f]; o->sum_phiDphi[f] = (double)GrD[f];
    }
    S ap = -p_a / (S(6) * S(V) * mpl * mpl);                                /* (2.14) */
    S H = ap / a2;
    o->a = (double)a; o->p_a = (double)p_a; o->eta = (double)eta;
    o->pot = (double)Vbar; o->rho = (double)rho; o->pressure = (double)P; o->hubble = (double)H;
    o->residual = std::isinf((double)mpl) ? 0.0 : (double)fabsl((long double)(rho / (S(3) * mpl * mpl * H * H) - S(1)));
    return ORACLE_OK;
  }

  int set_background(double a_in, double pa_in) override {
    if (!(a_in > 0) || !std::isfinite(a_in)) { err = "a must be finite and > 0"; return ORACLE_EINVAL; }
    a = S(a_in);
    if (std::isnan(pa_in)) {                                  /* reading G10: (2.18), expanding branch */
      if (!have_fields) { err = "p_a=NaN needs fields"; return ORACLE_ESTATE; }
      if (std::isinf((double)mpl)) { err = "p_a=NaN with static background"; return ORACLE_EINVAL; }
      S K[4], Gr[4], GrD[4], Vbar;
      averages(K, Gr, GrD, &Vbar);
      S a2 = a * a;
      S rho = Vbar + rho_g / (a2 * a2) + rho_m / (a2 * a);
      for (int f = 0; f < nf; ++f) rho += K[f] + Gr[f];
      if (!(rho >= 0)) { err = "negative energy density"; return ORACLE_EINVAL; }
      S ap = a2 * S(sqrtl((long double)(rho / S(3)))) / mpl;                /* (2.18) */
      p_a = -S(6) * S(V) * mpl * mpl * ap;                                  /* (2.11) */
    } else {
      p_a = S(pa_in);
    }
    return ORACLE_OK;
  }

  int set_dt(double d) override {
    if (d == 0 || !std::isfinite(d)) { err = "dt must be finite and non-zero"; return ORACLE_EINVAL; }
    dt = S(d);
    return ORACLE_OK;
  }

  int set_adaptive(int on) override { adaptive = on != 0; return ORACLE_OK; }

  int laplacian(int f, double* out) override {
    if (f < 0 || f >= nf || !out) { err = "bad field index"; return ORACLE_EINVAL; }
    for (int z = 0; z < N; ++z) for (int y = 0; y < N; ++y) for (int x = 0; x < N; ++x)
      out[((size_t)z * N + y) * N + x] = (double)lap(f, x, y, z);
    return ORACLE_OK;
  }
  int gradient_energy(int f, double* out) override {
    if (f < 0 || f >= nf || !out) { err = "bad field index"; return ORACLE_EINVAL; }
    for (int z = 0; z < N; ++z) for (int y = 0; y < N; ++y) for (int x = 0; x < N; ++x)
      out[((size_t)z * N + y) * N + x] = (double)grad_e(f, x, y, z);
    return ORACLE_OK;
  }
  int potential(const double* p_in, double* Vout, double* dVout) override {
    S p[4], dV[4];
    for (int f = 0; f < nf; ++f) p[f] = S(p_in[f]);
    S v = pot(p, dV);
    *Vout = (double)v;
    for (int f = 0; f < nf; ++f) dVout[f] = (double)dV[f];
    return ORACLE_OK;
  }
};

thread_local std::string g_create_err;

template <class T, class S, class IO>
Base* make(int N, double L, int nf, const oracle_params* mp, int order, double dt, const double* cs) {
  auto* s = new Stepper<T, S, IO>();
  s->N = N; s->nf = nf; s->order = order; s->V = (size_t)N * N * N;
  s->L = S(L); s->dx = S(L) / S(N); s->dt = S(dt);
  s->mpl = S(mp->mpl); s->rho_g = S(mp->rho_gamma0); s->rho_m = S(mp->rho_m0);
  s->a = 1; s->p_a = 0; s->eta = 0; s->model = mp->model;
  for (int i = 0; i < 8; ++i) s->par[i] = S(mp->p[i]);
  if (cs[0] == 0 && cs[1] == 0 && cs[2] == 0 && cs[3] == 0) {               /* reading G1 */
    s->c[0] = S(-128) / S(30); s->c[1] = S(14) / S(30); s->c[2] = S(3) / S(30); s->c[3] = S(1) / S(30);
  } else {
    for (int i = 0; i < 4; ++i) s->c[i] = S(cs[i]);
  }
  s->phi.assign((size_t)nf * s->V, T(0));
  s->pi.assign((size_t)nf * s->V, T(0));
  return s;
}

}  // namespace

struct oracle_ctx { Base* impl; };

extern "C" {

int oracle_create(oracle_ctx** out, int N, double L, int nfields, const oracle_params* mp, int order,
                  double dt) {
  if (!out) return ORACLE_EINVAL;
  *out = nullptr;
  if (!mp) return ORACLE_EINVAL;
  if (N < 3 || !(L > 0) || !std::isfinite(L)) return ORACLE_EINVAL;
  if (nfields < 1 || nfields > 4) return ORACLE_EINVAL;
  if (order != 2 && order != 4 && order != 6 && order != 8) return ORACLE_EINVAL;
  if (dt == 0 || !std::isfinite(dt)) return ORACLE_EINVAL;
  if (mp->model < ORACLE_FREE || mp->model > ORACLE_QBALL) return ORACLE_EINVAL;
  if ((mp->model == ORACLE_CHAOTIC || mp->model == ORACLE_QBALL) && nfields != 2) return ORACLE_EINVAL;
  if (mp->model == ORACLE_OSCILLON && nfields != 1) return ORACLE_EINVAL;
  if (!(mp->mpl > 0)) return ORACLE_EINVAL;                                  /* +INF allowed */
  if (mp->model == ORACLE_QBALL && !(mp->p[2] > 0)) return ORACLE_EINVAL;    /* M^2 > 0 */
  int prec = mp->precision == 0 ? 64 : mp->precision;
  if (prec != 32 && prec != 64 && prec != 80) return ORACLE_EINVAL;
  const double* cs = mp->stencil;
  if (!(cs[0] == 0 && cs[1] == 0 && cs[2] == 0 && cs[3] == 0)) {
    /* D must annihilate constants: c0 = -(6c1+12c2+8c3) (needed for (2.17)) */
    double s = 6 * cs[1] + 12 * cs[2] + 8 * cs[3];
    if (!(std::fabs(cs[0] + s) <= 1e-12 * (std::fabs(cs[0]) + std::fabs(s)))) return ORACLE_EINVAL;
  }
  try {
    Base* b = nullptr;
    if (prec == 32) b = make<float, double, float>(N, L, nfields, mp, order, dt, cs);
    else if (prec == 64) b = make<double, double, double>(N, L, nfields, mp, order, dt, cs);
    else b = make<long double, long double, double>(N, L, nfields, mp, order, dt, cs);
    *out = new oracle_ctx{b};
  } catch (const std::bad_alloc&) {
    return ORACLE_ENOMEM;
  }
  return ORACLE_OK;
}

int oracle_set_fields(oracle_ctx* c, const void* phi, const void* pi) { return c ? c->impl->set_fields(phi, pi) : ORACLE_EINVAL; }
int oracle_set_background(oracle_ctx* c, double a, double p_a) { return c ? c->impl->set_background(a, p_a) : ORACLE_EINVAL; }
int oracle_set_dt(oracle_ctx* c, double dt) { return c ? c->impl->set_dt(dt) : ORACLE_EINVAL; }
int oracle_set_adaptive(oracle_ctx* c, int on) { return c ? c->impl->set_adaptive(on) : ORACLE_EINVAL; }
int oracle_step(oracle_ctx* c, int n) { return c ? c->impl->step(n) : ORACLE_EINVAL; }
int oracle_read_fields(oracle_ctx* c, void* phi, void* pi) { return c ? c->impl->read_fields(phi, pi) : ORACLE_EINVAL; }
int oracle_energies(oracle_ctx* c, oracle_energy* o) { return c ? c->impl->energies(o) : ORACLE_EINVAL; }
int oracle_destroy(oracle_ctx* c) { if (!c) return ORACLE_EINVAL; delete c->impl; delete c; return ORACLE_OK; }
const char* oracle_last_error(const oracle_ctx* c) { return c ? c->impl->err.c_str() : "null context"; }

int oracle_stage_weights(int order, double* w, int cap) {
  long double t[16];
  int s = stage_weights(order, t);
  if (s == 0 || s > cap) return 0;
  for (int i = 0; i < s; ++i) w[i] = (double)t[i];
  return s;
}
int oracle_laplacian(oracle_ctx* c, int f, double* out) { return c ? c->impl->laplacian(f, out) : ORACLE_EINVAL; }
int oracle_gradient_energy(oracle_ctx* c, int f, double* out) { return c ? c->impl->gradient_energy(f, out) : ORACLE_EINVAL; }
int oracle_potential(oracle_ctx* c, const double* phi, double* V, double* dV) { return c ? c->impl->potential(phi, V, dV) : ORACLE_EINVAL; }

}  // extern "C"
