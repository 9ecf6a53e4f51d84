"""Oracle for the linearised solver of arXiv 1201.5029 section 2.2.  TEST INFRASTRUCTURE ONLY.

What it computes.  The fields are split into a homogeneous background and perturbations,
phi_i(x) = phi_{0,i} + dphi_i(x) (2.21); the background (a, p_a, phi_0, pi_0) follows (2.35)-(2.36) on its own, the
perturbations follow the linear equations (2.37), evolved in Fourier space (2.38), where modes do not couple:

    a'      = -p_a / (6 V_L mpl^2)                                                          (2.35)
    p_a'    = V_L ( sum_i pi_{0,i}^2 / a^3 - 4 a^3 V(phi_0) ) - V_L rho_m0                  (2.35), (2.20)
    phi_0'  = pi_0 / a^2 ,   pi_0' = -a^4 dV/dphi_0                                         (2.36)
    dPhi_k' = dPi_k / a^2                                                                   (2.38)
    dPi_k'  = -k_eff^2 a^2 dPhi_k / dx^2 - a^4 sum_j V_ij(phi_0) dPhi_{j,k}                 (2.38), (2.26)

with V_ij = d^2 V / dphi_i dphi_j at the background (dV^(2)/d(dphi_i) = sum_j V_ij dphi_j, check with (2.27)) and
-k_eff^2 the eigenvalue of the stencil D of (2.7) on the mode.  The Hamiltonian splits into five integrable parts
(2.49), composed to second order as (2.50)
    Phi2(h) = H1(h/2) H2(h/2) H3(h/2) H4(h/2) H5(h) H4(h/2) H3(h/2) H2(h/2) H1(h/2)
      H1(e): a   -= p_a / (6 V_L mpl^2) e
      H2(e): p_a += (V_L sum_i pi_0^2 / a^3 - V_L rho_m0) e ;  phi_0 += pi_0 / a^2 e
      H3(e): p_a += -4 a^3 V_L V(phi_0) e ;  pi_0 += -a^4 dV/dphi_0 e
      H4(e): dPhi += dPi / a^2 e
      H5(e): dPi_i += (-k_eff^2 a^2 / dx^2 dPhi_i - a^4 sum_j V_ij(phi_0) dPhi_j) e
and to order 4/6/8 with the same stage weights as the non-linear step ((2.43)-(2.45), Table 1).  The composition is
palindromic, so the operator-ordering convention is immaterial.

Two ways to advance the perturbations, which must agree to rounding:
  step(n)            every Fourier mode evolved on its own ("naive version");
  growth_step(n)     the linear map M(tau, k_eff^2) of (2.51) evolved once per DISTINCT value of k_eff^2 (columns
                     M 1_i started from unit vectors), then every mode multiplied by the matrix of its k_eff^2.

Readings (G25-G28):
  G25  (2.35) prints "sum_i V_L a^3 (pi_0^2/a^6 - 4 V)": the sum runs over the kinetic term only, V is one function
       of all fields -- as in (2.47) restricted to a homogeneous lattice; the rho_m0 term of (2.20) is kept.
  G26  (2.32)/(2.34) are inconsistent by a factor V_L (pi_0 = a^2 phi_0' is a per-site momentum, the Hamiltonian sums
       V_L copies); the equations of motion (2.35)-(2.36) as printed are what is integrated.
  G27  (2.22): the k = 0 mode of the perturbations is removed on input and stays exactly zero (its equation is the
       background's).
  G28  "distinct values of k_eff^2": k_eff^2(n) is a symmetric function of (cos 2 pi n_x/N, ..), so modes are grouped
       by the sorted triple (|n|_(1) <= |n|_(2) <= |n|_(3)), |n_i| <= N/2: (M+1)(M+2)(M+3)/6 classes, M = floor(N/2).
       Accidental coincidences of k_eff^2 between different triples are not merged (harmless).

Plain numpy, fp64 (longdouble on request), vectorised over modes, one Python loop over stages; the FFT is numpy's.
Shares no code with the CUDA path.  Pins: tests/test_oracle_linear.py.
"""
import math

import numpy as np

FREE, CHAOTIC, OSCILLON, QBALL = 0, 1, 2, 3

_T6 = ("0.78451361047755726382", "0.23557321335935813368", "-1.17767998417887100695")
_T8 = ("0.74167036435061295345", "-0.40910082580003159400", "0.19075471029623837995", "-0.57386247111608226666",
       "0.29906418130365592384", "0.33462491824529818378", "0.31529309239676659663")


def stage_weights(order, dtype=np.float64):
    """(2.42); (2.43)-(2.44) with n = 1 (reading G2); Table 1, symmetric, summing to one."""
    ld = np.longdouble
    if order == 2:
        w = [ld(1)]
    elif order == 4:
        c = ld(2) ** (ld(1) / ld(3))
        w = [ld(1) / (ld(2) - c), -c / (ld(2) - c), ld(1) / (ld(2) - c)]
    elif order in (6, 8):
        half = [ld(t) for t in (_T6 if order == 6 else _T8)]
        mid = ld(1) - ld(2) * sum(half, ld(0))
        w = half + [mid] + half[::-1]
    else:
        raise ValueError("order must be 2, 4, 6 or 8")
    return [dtype(x) for x in w]


def potential(model, p, mpl, phi):
    """V, dV/dphi_i and the Hessian V_ij at the homogeneous point phi (sequence of nf numbers).
    (3.2) PAPER.md:427, (3.3) PAPER.md:456, (3.4) PAPER.md:481 with readings G6-G8."""
    phi = [x for x in phi]
    nf = len(phi)
    T = type(phi[0])
    H = [[T(0)] * nf for _ in range(nf)]
    if model == FREE:
        V = sum(T(0.5) * T(p[f]) * phi[f] * phi[f] for f in range(nf))
        dV = [T(p[f]) * phi[f] for f in range(nf)]
        for f in range(nf):
            H[f][f] = T(p[f])
    elif model == CHAOTIC:
        m2, g2 = T(p[0]), T(p[1])
        ph, ch = phi
        V = T(0.5) * m2 * ph * ph + T(0.5) * g2 * ph * ph * ch * ch
        dV = [m2 * ph + g2 * ph * ch * ch, g2 * ph * ph * ch]
        H = [[m2 + g2 * ch * ch, T(2) * g2 * ph * ch], [T(2) * g2 * ph * ch, g2 * ph * ph]]       # (2.27)
    elif model == OSCILLON:
        m2, lam, g6 = T(p[0]), T(p[1]), T(p[2])
        ph = phi[0]
        p2 = ph * ph
        V = T(0.5) * m2 * p2 - lam / T(4) * p2 * p2 + g6 / T(6) * p2 * p2 * p2
        dV = [m2 * ph - lam * p2 * ph + g6 * p2 * p2 * ph]
        H = [[m2 - T(3) * lam * p2 + T(5) * g6 * p2 * p2]]
    elif model == QBALL:
        m2, K, M2, l6 = T(p[0]), T(p[1]), T(p[2]), T(p[3])
        six = l6 / (T(mpl) * T(mpl)) if math.isfinite(float(mpl)) else T(0)
        r2 = (phi[0] * phi[0] + phi[1] * phi[1]) / T(2)
        tiny = float(r2) < 2.2250738585072014e-308
        lg = T(0) if tiny else T(np.log(r2 / M2))
        common = m2 * (T(1) + K + K * lg) + T(3) * six * r2 * r2
        V = m2 * r2 * (T(1) + K * lg) + six * r2 * r2 * r2
        dV = [common * phi[0], common * phi[1]]
        # d common / d phi_j = (m2 K / r2 + 6 six r2) phi_j   (d r2 / d phi_j = phi_j)
        dc = T(0) if tiny else m2 * K / r2 + T(6) * six * r2
        H = [[common * (T(1) if i == j else T(0)) + dc * phi[i] * phi[j] for j in range(nf)] for i in range(nf)]
    else:
        raise ValueError("unknown model")
    return V, dV, H


def k_eff2_of(n, N, stencil, dtype=np.float64):
    """k_eff^2 >= 0 of integer wave vectors n[..., 3]: minus the eigenvalue of (2.7)."""
    c0, c1, c2, c3 = (dtype(c) for c in stencil)
    C = np.cos(dtype(2) * dtype(math.pi) * np.asarray(n, dtype=dtype) / dtype(N))
    Cx, Cy, Cz = C[..., 0], C[..., 1], C[..., 2]
    return -(c0 + 2 * c1 * (Cx + Cy + Cz) + 4 * c2 * (Cx * Cy + Cy * Cz + Cz * Cx) + 8 * c3 * Cx * Cy * Cz)


def distinct_table(N):
    """Reading G28.  Returns (triples [T,3] sorted ascending within each row, index [N,N,N] mapping the mode
    (iz, iy, ix) to its row, multiplicity [T])."""
    M = N // 2
    fold = np.minimum(np.arange(N), N - np.arange(N))             # |n_i| in 0..M
    iz, iy, ix = np.meshgrid(fold, fold, fold, indexing="ij")
    s = np.sort(np.stack([iz, iy, ix], axis=-1), axis=-1)          # (lo, mid, hi)
    key = (s[..., 2] * (M + 1) + s[..., 1]) * (M + 1) + s[..., 0]
    uniq, index = np.unique(key.ravel(), return_inverse=True)
    triples = np.stack([uniq % (M + 1), (uniq // (M + 1)) % (M + 1), uniq // (M + 1) ** 2], axis=-1)
    mult = np.bincount(index, minlength=len(uniq))
    return triples, index.reshape(N, N, N), mult


class LinearOracle:
    def __init__(self, N, L, nfields, model, p=(), order=4, dt=0.01, mpl=1.0, rho_gamma0=0.0, rho_m0=0.0,
                 stencil=(0, 0, 0, 0), precision=64):
        self.T = np.longdouble if precision == 80 else np.float64
        T = self.T
        self.N, self.nf, self.model, self.p, self.order = N, nfields, model, tuple(p), order
        self.L, self.dx, self.dt, self.mpl = T(L), T(L) / T(N), T(dt), T(mpl)
        self.rho_g, self.rho_m = T(rho_gamma0), T(rho_m0)
        self.VL = T(N) ** 3
        if all(c == 0 for c in stencil):
            stencil = (T(-128) / T(30), T(14) / T(30), T(3) / T(30), T(1) / T(30))              # reading G1
        self.stencil = tuple(T(c) for c in stencil)
        self.w = stage_weights(order, T)
        self.a, self.p_a, self.eta = T(1), T(0), T(0)
        self.phi0, self.pi0 = [T(0)] * nfields, [T(0)] * nfields
        fold = np.arange(N)
        fold = np.where(fold <= N // 2, fold, fold - N)
        nz, ny, nx = np.meshgrid(fold, fold, fold, indexing="ij")
        self.k2 = k_eff2_of(np.stack([nx, ny, nz], axis=-1), N, self.stencil, T)                  # [N,N,N]
        ctype = np.clongdouble if precision == 80 else np.complex128
        self.dPhi = np.zeros((nfields, N, N, N), ctype)
        self.dPi = np.zeros((nfields, N, N, N), ctype)

    # ------------------------------------------------------------------ state
    def set_background(self, a, p_a, phi0, pi0):
        """p_a = NaN: first Friedmann equation (2.18) on the background alone, expanding branch (reading G10):
        rho = sum pi_0^2/(2 a^6) + V(phi_0) + rho_g/a^4 + rho_m/a^3, p_a = -6 V_L mpl a^2 sqrt(rho/3)."""
        T = self.T
        self.a = T(a)
        self.phi0, self.pi0 = [T(x) for x in phi0], [T(x) for x in pi0]
        if math.isnan(float(p_a)):
            rho = self.background_energy()["rho"]
            self.p_a = -T(6) * self.VL * self.mpl * self.a * self.a * np.sqrt(rho / T(3))
        else:
            self.p_a = T(p_a)

    def set_perturbations(self, dphi, dpi):
        """Real-space perturbations [nf, N, N, N] (z, y, x) -> Fourier space (plain DFT sum_x f exp(-2 pi i n.x/N));
        the k = 0 mode is removed (2.22), reading G27."""
        dt = np.float64 if self.T is np.float64 else np.longdouble
        self.dPhi = np.fft.fftn(np.asarray(dphi, dtype=dt), axes=(1, 2, 3)).astype(self.dPhi.dtype)
        self.dPi = np.fft.fftn(np.asarray(dpi, dtype=dt), axes=(1, 2, 3)).astype(self.dPi.dtype)
        self.dPhi[:, 0, 0, 0] = 0
        self.dPi[:, 0, 0, 0] = 0

    def read_perturbations(self):
        f = lambda F: np.real(np.fft.ifftn(F.astype(np.complex128), axes=(1, 2, 3)))
        return f(self.dPhi), f(self.dPi)

    def background_energy(self):
        T = self.T
        V, _, _ = potential(self.model, self.p, self.mpl, self.phi0)
        a2 = self.a * self.a
        K = sum(q * q for q in self.pi0) / (T(2) * a2 * a2 * a2)
        rho = K + V + self.rho_g / (a2 * a2) + self.rho_m / (a2 * self.a)
        ap = -self.p_a / (T(6) * self.VL * self.mpl * self.mpl)
        H = ap / a2
        res = abs(rho / (T(3) * self.mpl * self.mpl * H * H) - T(1)) if math.isfinite(float(self.mpl)) and H != 0 else T(0)
        return {"a": self.a, "p_a": self.p_a, "eta": self.eta, "kin": K, "pot": V, "rho": rho, "hubble": H,
                "residual": res}

    # ------------------------------------------------------------------ the five flows of (2.49)
    def _H1(self, e):
        self.a = self.a - self.p_a / (self.T(6) * self.VL * self.mpl * self.mpl) * e

    def _H2(self, e):
        a = self.a
        s = sum(q * q for q in self.pi0)
        self.p_a = self.p_a + (self.VL * s / (a * a * a) - self.VL * self.rho_m) * e
        self.phi0 = [f + q / (a * a) * e for f, q in zip(self.phi0, self.pi0)]

    def _H3(self, e):
        a = self.a
        V, dV, _ = potential(self.model, self.p, self.mpl, self.phi0)
        self.p_a = self.p_a + (-self.T(4) * a * a * a * self.VL * V) * e
        self.pi0 = [q - a * a * a * a * d * e for q, d in zip(self.pi0, dV)]

    def _H4(self, e, Phi, Pi):
        Phi += Pi * (e / (self.a * self.a))

    def _H5(self, e, Phi, Pi, k2):
        a = self.a
        _, _, Hs = potential(self.model, self.p, self.mpl, self.phi0)
        kD = a * a / (self.dx * self.dx)
        a4 = a * a * a * a
        new = []
        for i in range(self.nf):
            force = -(k2 * kD) * Phi[i]
            for j in range(self.nf):
                force = force - a4 * Hs[i][j] * Phi[j]
            new.append(force * e)
        for i in range(self.nf):
            Pi[i] += new[i]

    def _phi2(self, h, Phi, Pi, k2):
        T = self.T
        e = h / T(2)
        self._H1(e); self._H2(e); self._H3(e); self._H4(e, Phi, Pi)
        self._H5(h, Phi, Pi, k2)
        self._H4(e, Phi, Pi); self._H3(e); self._H2(e); self._H1(e)

    def _advance(self, n, Phi, Pi, k2):
        for _ in range(n):
            for w in self.w:
                self._phi2(w * self.dt, Phi, Pi, k2)
            self.eta = self.eta + self.dt

    # ------------------------------------------------------------------ public evolution
    def step(self, n=1):
        """Every Fourier mode evolved on its own (the paper's "naive version")."""
        self._advance(n, self.dPhi, self.dPi, self.k2)

    def growth_matrices(self, n):
        """Advance the BACKGROUND n steps and return (M [T, 2nf, 2nf], index [N,N,N]): M[t] maps
        (dPhi_1, dPi_1, .., dPhi_nf, dPi_nf) at the start to the same vector n steps later for every mode of class t
        (2.51).  Column c of M is the evolution of the unit vector 1_c."""
        nf, T = self.nf, self.T
        triples, index, _ = distinct_table(self.N)
        k2 = k_eff2_of(triples, self.N, self.stencil, T)                                         # [Tn]
        Tn = len(k2)
        # 2 nf unit vectors per class: Phi[i] has shape [Tn, 2 nf] (one column per initial unit vector)
        Phi = np.zeros((nf, Tn, 2 * nf), T)
        Pi = np.zeros((nf, Tn, 2 * nf), T)
        for i in range(nf):
            Phi[i, :, 2 * i] = 1
            Pi[i, :, 2 * i + 1] = 1
        self._advance(n, Phi, Pi, k2[:, None])
        M = np.zeros((Tn, 2 * nf, 2 * nf), T)
        for i in range(nf):
            M[:, 2 * i, :] = Phi[i]
            M[:, 2 * i + 1, :] = Pi[i]
        return M, index

    def growth_step(self, n=1):
        """n steps through the growth matrices (2.51): background advanced once, one matrix per distinct k_eff^2
        class, every mode multiplied by its class's matrix."""
        M, index = self.growth_matrices(n)
        nf = self.nf
        vec = np.empty((2 * nf,) + self.dPhi.shape[1:], self.dPhi.dtype)
        for i in range(nf):
            vec[2 * i], vec[2 * i + 1] = self.dPhi[i], self.dPi[i]
        Mk = M[index]                                                                             # [N,N,N,2nf,2nf]
        out = np.einsum("zyxrc,czyx->rzyx", Mk, vec)
        for i in range(nf):
            self.dPhi[i], self.dPi[i] = out[2 * i], out[2 * i + 1]
