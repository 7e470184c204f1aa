"""Brute-force full-grid 6D Vlasov-Poisson solvers for tiny grids (n = 4 per dimension), used ONLY to pin
the oracle (tests/test_oracle_bruteforce.py).  Written independently of oracle/ (no import of it): they
work on the full array F[x3, x2, x1, v3, v2, v1] and know nothing about low-rank factors.

* `Mirrored`: applies to F itself the sequence of flows of Algorithm 2 with the
  sub-flows of section 4.  At full rank (r = N_x = N_v) the projectors P_X, P_V of
  eqs. (3)-(5) are the identity, so the DLR integrator and this solver are the same
  map up to rounding: K step = dF/dt = -v.grad_x F + E.grad_v F solved with x-Fourier sub-flows,
  S step = dF/dt = +v.grad_x F - E.grad_v F by RK4, L step = the K equation solved with v-Fourier
  sub-flows.
* `classical_strang`: the textbook Strang splitting (x-advection tau/2, Poisson, v-advection tau,
  x-advection tau/2) with exact Fourier shifts - an independent second-order solver of the same
  semi-discrete problem.
"""
import math
import numpy as np


def _phi1(z):
    z = np.asarray(z, dtype=complex)
    zz = np.where(z == 0, 1.0, z)
    return np.where(z == 0, 1.0, np.expm1(zz) / zz)


def _phi2(z):
    """(e^z - 1 - z)/z^2 in extended precision by its power series (|z| small) or directly"""
    z = np.asarray(z, dtype=np.clongdouble)
    out = np.zeros(z.shape, dtype=np.clongdouble)
    term = np.full(z.shape, 0.5, dtype=np.clongdouble)
    for m in range(0, 60):
        out = out + term
        term = term * z / (m + 3)
    zz = np.where(np.abs(z) < 2.0, 1.0, z)
    direct = (np.exp(zz) - 1.0 - zz) / (zz * zz)
    return np.where(np.abs(z) < 2.0, out, direct).astype(complex)


class Mirrored:
    def __init__(self, n, x_lo, x_hi, v_lo, v_hi):
        self.n = n
        self.hx = (x_hi - x_lo) / n
        self.hv = (v_hi - v_lo) / n
        self.v = v_lo + self.hv * np.arange(n)
        m = np.fft.fftfreq(n, 1.0 / n)
        mt = m.copy()
        mt[n // 2] = 0.0                       # odd-derivative wavenumber is zero at Nyquist
        self.kx_true = 2 * math.pi * m / (x_hi - x_lo)
        self.kx = 2 * math.pi * mt / (x_hi - x_lo)
        self.kv = 2 * math.pi * mt / (v_hi - v_lo)

    # axis helpers: x_d lives on axis 2-d, v_d on axis 5-d
    def _ax(self, vec, axis):
        s = [1] * 6
        s[axis] = self.n
        return np.asarray(vec).reshape(s)

    def dx(self, F, d):
        ax = 2 - d
        return np.fft.ifft(1j * self._ax(self.kx, ax) * np.fft.fft(F, axis=ax), axis=ax).real

    def dv(self, F, d):
        ax = 5 - d
        return np.fft.ifft(1j * self._ax(self.kv, ax) * np.fft.fft(F, axis=ax), axis=ax).real

    def field(self, F):
        n = self.n
        rho = -(self.hv ** 3) * F.sum(axis=(3, 4, 5))
        rh = np.fft.fftn(rho)
        k2 = (self.kx_true.reshape(n, 1, 1) ** 2 + self.kx_true.reshape(1, n, 1) ** 2
              + self.kx_true.reshape(1, 1, n) ** 2)
        k2[0, 0, 0] = 1.0
        ph = rh / k2
        ph[0, 0, 0] = 0.0
        E = []
        for d in range(3):
            s = [1, 1, 1]
            s[2 - d] = n
            E.append(np.fft.ifftn(-1j * self.kx.reshape(s) * ph).real)
        return E                                # E[d][x3, x2, x1]

    def electric_energy(self, F):
        E = self.field(F)
        return 0.5 * self.hx ** 3 * sum(np.sum(e * e) for e in E)

    def mass(self, F):
        return self.hx ** 3 * self.hv ** 3 * F.sum()

    def _Ex(self, E, d):
        return E[d].reshape(self.n, self.n, self.n, 1, 1, 1)

    # ---- K flow: Fourier in x ----
    def K_flow(self, F, t, E, order):
        fx = lambda A: np.fft.fftn(A, axes=(0, 1, 2))
        ifx = lambda A: np.fft.ifftn(A, axes=(0, 1, 2))

        def sub(Fh, d, tt):
            return Fh * np.exp(-1j * tt * self._ax(self.kx, 2 - d) * self._ax(self.v, 5 - d))

        def nonlin(A):
            return sum(self._Ex(E, d) * self.dv(A, d) for d in range(3))

        def third(Fh, tt, ordr):
            z = -1j * tt * self._ax(self.kx, 0) * self._ax(self.v, 3)
            G0 = fx(nonlin(ifx(Fh).real))
            a = np.exp(z) * Fh + tt * _phi1(z) * G0
            if ordr == 1:
                return a
            G1 = fx(nonlin(ifx(a).real))
            return a + tt * _phi2(z) * (G1 - G0)

        Fh = fx(F)
        if order == 1:
            Fh = third(sub(sub(Fh, 0, t), 1, t), t, 1)
        else:
            Fh = sub(sub(Fh, 0, t / 2), 1, t / 2)
            Fh = third(Fh, t, 2)
            Fh = sub(sub(Fh, 1, t / 2), 0, t / 2)
        return ifx(Fh).real

    # ---- L flow: Fourier in v ----
    def L_flow(self, F, t, E, order):
        fv = lambda A: np.fft.fftn(A, axes=(3, 4, 5))
        ifv = lambda A: np.fft.ifftn(A, axes=(3, 4, 5))

        def sub(Fh, d, tt):
            return Fh * np.exp(+1j * tt * self._ax(self.kv, 5 - d) * self._Ex(E, d))

        def nonlin(A):
            return -sum(self._ax(self.v, 5 - d) * self.dx(A, d) for d in range(3))

        def third(Fh, tt, ordr):
            z = +1j * tt * self._ax(self.kv, 3) * self._Ex(E, 2)
            G0 = fv(nonlin(ifv(Fh).real))
            a = np.exp(z) * Fh + tt * _phi1(z) * G0
            if ordr == 1:
                return a
            G1 = fv(nonlin(ifv(a).real))
            return a + tt * _phi2(z) * (G1 - G0)

        Fh = fv(F)
        if order == 1:
            Fh = third(sub(sub(Fh, 0, t), 1, t), t, 1)
        else:
            Fh = sub(sub(Fh, 0, t / 2), 1, t / 2)
            Fh = third(Fh, t, 2)
            Fh = sub(sub(Fh, 1, t / 2), 0, t / 2)
        return ifv(Fh).real

    # ---- S flow: RK4 on the backward equation ----
    def S_flow(self, F, t, E):
        def rhs(A):
            return sum(self._ax(self.v, 5 - d) * self.dx(A, d) - self._Ex(E, d) * self.dv(A, d)
                       for d in range(3))
        k1 = rhs(F)
        k2 = rhs(F + 0.5 * t * k1)
        k3 = rhs(F + 0.5 * t * k2)
        k4 = rhs(F + t * k3)
        return F + (t / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)

    def step_alg1(self, F, tau):
        E0 = self.field(F)
        F = self.K_flow(F, tau, E0, 1)
        F = self.S_flow(F, tau, E0)
        return self.L_flow(F, tau, E0, 1)

    def step_alg2(self, F, tau):
        Eh = self.field(self.step_alg1(F, tau / 2))
        F = self.K_flow(F, tau / 2, Eh, 2)
        F = self.S_flow(F, tau / 2, Eh)
        F = self.L_flow(F, tau, Eh, 2)
        F = self.S_flow(F, tau / 2, Eh)
        return self.K_flow(F, tau / 2, Eh, 2)

    # ---- independent classical Strang splitting ----
    def classical_strang(self, F, tau):
        def xadv(A, t):
            ph = sum(self._ax(self.kx, 2 - d) * self._ax(self.v, 5 - d) for d in range(3))
            return np.fft.ifftn(np.exp(-1j * t * ph) * np.fft.fftn(A, axes=(0, 1, 2)), axes=(0, 1, 2)).real

        def vadv(A, t, E):
            ph = sum(self._ax(self.kv, 5 - d) * self._Ex(E, d) for d in range(3))
            return np.fft.ifftn(np.exp(+1j * t * ph) * np.fft.fftn(A, axes=(3, 4, 5)), axes=(3, 4, 5)).real

        F = xadv(F, tau / 2)
        F = vadv(F, tau, self.field(F))
        return xadv(F, tau / 2)
