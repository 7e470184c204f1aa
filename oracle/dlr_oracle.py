"""CPU ORACLE (test infrastructure, not the product) for the second-order projector-splitting
dynamical low-rank (DLR) integrator of the 6D Vlasov-Poisson system, written from
Cassini & Einkemmer, arXiv 2110.13481 (cited below as PAPER.md:<line>, section/equation).

* plain NumPy, fp64 (the paper computes in double precision), no blocking, no fusion:
  every function follows the paper's equations in the paper's order and notation so that it can be
  checked against the paper by eye;  library primitives used as steps: numpy.fft (3D DFT), matmul.
* shares NO code with the CUDA path (paper_2110_13481_b200/); only tests/, __graft_entry__.smoke()
  and bench.py's cpu_baseline / --impl reference legs may import this module.
* readings of the paper where it is silent (R1..R16) are those listed in DESIGN.md section 3.
* pins (tests/test_oracle_*.py, all run with -m "not gpu"): naive-DFT/closed-form checks of the
  discretisation, n=4 full-rank agreement with a brute-force 6D solver, second-order convergence to an
  independent Strang solver, exact free streaming of the K-flow, Landau damping rate; step_bug (the unconventional
  integrator the paper names): full-rank agreement with a brute-force forward RK4 step, first-order
  convergence to the limit of Algorithm 2, robustness to a rank-deficient S (tests/test_oracle_bug.py).
  Parity unpinned: the choice among equally valid second-order variants (R8 which exponential RK,
  R10 order of directions) is pinned only up to "the brute-force solver that uses the same choice
  agrees, and the scheme converges at order 2"; results at rank r < 7 depend on the random padding.

Layout: a factor is an (N, r) array, row index I = i1 + n1*(i2 + n2*i3) (x1 fastest, PAPER.md:282
"degrees of freedom are linearised"; the ordering itself is reading R1).
"""
import math
import numpy as np


# --------------------------------------------------------------------------------------
# grid, DFT conventions, wavenumbers                                  (readings R1, R3, R4)
# --------------------------------------------------------------------------------------
class Grid3:
    """Uniform periodic left-closed grid on [lo, hi)^3: x_d(i) = lo_d + i*h_d, i = 0..n_d-1
    ("number of discretization points, the left extremes ... and the grid spacing";
    PAPER.md:452 periodic in all directions).  Quadrature weight is the constant h1*h2*h3
    (Fig. 2 inner_product_from_const_weight)."""

    def __init__(self, n, lo, hi):
        self.n = tuple(int(a) for a in n)            # (n1, n2, n3)
        self.lo = tuple(float(a) for a in lo)
        self.hi = tuple(float(a) for a in hi)
        self.h = tuple((self.hi[d] - self.lo[d]) / self.n[d] for d in range(3))
        self.N = self.n[0] * self.n[1] * self.n[2]
        self.w = self.h[0] * self.h[1] * self.h[2]   # h^3
        self.shape = (self.n[2], self.n[1], self.n[0])   # numpy shape of one column: (i3, i2, i1)

    def _bcast(self, a, d):
        s = [1, 1, 1]
        s[2 - d] = self.n[d]
        return np.asarray(a).reshape(s)

    def coord(self, d):
        """grid coordinate d (0-based) broadcastable against an (n3, n2, n1) array"""
        return self._bcast(self.lo[d] + self.h[d] * np.arange(self.n[d]), d)

    def coord_flat(self, d):
        return np.broadcast_to(self.coord(d), self.shape).reshape(-1)

    def m(self, d):
        """integer DFT wavenumbers 0,1,..,n/2-1,-n/2,..,-1"""
        n = self.n[d]
        i = np.arange(n)
        return np.where(i < (n + 1) // 2, i, i - n)

    def k(self, d):
        """true wavenumber 2*pi*m/L (used in the Laplacian symbol, R4)"""
        L = self.hi[d] - self.lo[d]
        return self._bcast(2.0 * math.pi * self.m(d) / L, d)

    def kt(self, d):
        """odd-derivative wavenumber: as k but 0 at the Nyquist index n/2 (R4)"""
        n = self.n[d]
        L = self.hi[d] - self.lo[d]
        m = self.m(d).astype(float)
        if n % 2 == 0:
            m[n // 2] = 0.0
        return self._bcast(2.0 * math.pi * m / L, d)


def to_grid(A, g):
    """(N, r) factor -> (r, n3, n2, n1) array of its columns on the grid"""
    return np.ascontiguousarray(A.T).reshape((A.shape[1],) + g.shape)


def to_mat(Ag):
    """(r, n3, n2, n1) -> (N, r)"""
    return Ag.reshape(Ag.shape[0], -1).T.copy()


def fft3(Ag):
    """forward DFT of every column, exp(-2 pi i m j / n) per dimension, unnormalised (R3)"""
    return np.fft.fftn(Ag, axes=(-3, -2, -1))


def ifft3(Ah):
    """inverse DFT (1/n per dimension)"""
    return np.fft.ifftn(Ah, axes=(-3, -2, -1))


def deriv(Ag, g, d):
    """spectral derivative d/dx_d: F^-1( i kt_d F(A) )   ("D^F")"""
    return ifft3(1j * g.kt(d) * fft3(Ag)).real


# --------------------------------------------------------------------------------------
# coefficients
# --------------------------------------------------------------------------------------
def coeff(A, Bm, w):
    """Ensign's coeff: A^T diag(w) B  (Fig. 1 line 8)"""
    return A.T @ (w[:, None] * Bm)


def coeff_C(V, gv):
    """C1_i = V^T diag(h_v^3 v_i) V,  C2_i = V^T diag(h_v^3) d_{v_i}V  (R2),
    rho_tilde = V^T omega_v with omega_v = h_v^3 * 1  (eq. (12))."""
    Vg = to_grid(V, gv)
    ones = np.ones(gv.N)
    C1 = [coeff(V, V, gv.w * gv.coord_flat(d)) for d in range(3)]
    C2 = [coeff(V, to_mat(deriv(Vg, gv, d)), gv.w * ones) for d in range(3)]
    rho_t = V.T @ (gv.w * ones)
    return C1, C2, rho_t


def coeff_D(X, E, gx):
    """D1_i = X^T diag(h_x^3 E_i) X,  D2_i = X^T diag(h_x^3) d_{x_i}X  (R2)."""
    Xg = to_grid(X, gx)
    ones = np.ones(gx.N)
    D1 = [coeff(X, X, gx.w * E[d]) for d in range(3)]
    D2 = [coeff(X, to_mat(deriv(Xg, gx, d)), gx.w * ones) for d in range(3)]
    return D1, D2


# --------------------------------------------------------------------------------------
# electric field                                  (eq. (1); (12),(13) :180-190)
# --------------------------------------------------------------------------------------
def field(A, p, gx, e_scale=1.0):
    """rho = -A p ;  -Laplace(phi) = rho + 1 ;  E = -grad(phi), all by DFT.
    (12): A = K, p = rho_tilde = V^T omega_v;   (13): A = X, p = L^T omega_v.
    The '+1' background only touches the k = 0 mode, which is dropped (R6).
    Laplacian symbol |k|^2 with the true wavenumbers, gradient with kt (R4).
    Returns E as a (3, N_x) array."""
    rho = -(A @ p)
    rho_h = np.fft.fftn(rho.reshape(gx.shape))
    k2 = gx.k(0) ** 2 + gx.k(1) ** 2 + gx.k(2) ** 2
    k2[0, 0, 0] = 1.0
    phi_h = rho_h / k2
    phi_h[0, 0, 0] = 0.0
    E = np.empty((3, gx.N))
    for d in range(3):
        E[d] = e_scale * np.fft.ifftn(-1j * gx.kt(d) * phi_h).real.reshape(-1)
    return E


# --------------------------------------------------------------------------------------
# small dense: Jacobi eigen-solver, phi functions, modified Gram-Schmidt
# --------------------------------------------------------------------------------------
def jacobi_eigh(M):
    """cyclic Jacobi for a symmetric matrix: M = T diag(lam) T^T  ("it is possible to
    diagonalize them"; the solver is not specified, the result enters only through T f(lam) T^T)."""
    A = 0.5 * (M + M.T)                       # R5: symmetrise before the eigen-solve
    n = A.shape[0]
    T = np.eye(n)
    normA = math.sqrt(np.sum(A * A))
    for _sweep in range(100):
        off = math.sqrt(np.sum(np.triu(A, 1) ** 2))
        if off <= 1e-16 * normA or off == 0.0:
            break
        for p in range(n - 1):
            for q in range(p + 1, n):
                apq = A[p, q]
                if abs(apq) <= 1e-20 * normA:
                    A[p, q] = A[q, p] = 0.0 if abs(apq) < 1e-300 else apq
                    continue
                theta = (A[q, q] - A[p, p]) / (2.0 * apq)
                if abs(theta) > 1e150:
                    t = 0.5 / theta
                else:
                    t = (1.0 if theta >= 0 else -1.0) / (abs(theta) + math.sqrt(theta * theta + 1.0))
                c = 1.0 / math.sqrt(t * t + 1.0)
                s = t * c
                Ap = A[:, p].copy()
                Aq = A[:, q].copy()
                A[:, p] = c * Ap - s * Aq
                A[:, q] = s * Ap + c * Aq
                Ap = A[p, :].copy()
                Aq = A[q, :].copy()
                A[p, :] = c * Ap - s * Aq
                A[q, :] = s * Ap + c * Aq
                A[p, q] = A[q, p] = 0.0
                Tp = T[:, p].copy()
                Tq = T[:, q].copy()
                T[:, p] = c * Tp - s * Tq
                T[:, q] = s * Tp + c * Tq
    return np.diag(A).copy(), T


_FACT = [math.factorial(i) for i in range(26)]


def phi1_imag(theta):
    """phi1(i theta) = (e^{i theta} - 1)/(i theta) = sin(theta)/theta + i (1 - cos(theta))/theta;
    Taylor series sum (i theta)^m/(m+1)! for |theta| < 1 (R7)."""
    theta = np.asarray(theta, dtype=float)
    small = np.abs(theta) < 1.0
    th = np.where(small, 1.0, theta)
    big = np.sin(th) / th + 1j * (2.0 * np.sin(0.5 * th) ** 2) / th
    ser = np.zeros(theta.shape, dtype=complex)
    z = 1j * np.where(small, theta, 0.0)
    for m in range(21, -1, -1):
        ser = ser * z + 1.0 / _FACT[m + 1]
    return np.where(small, ser, big)


def phi2_imag(theta):
    """phi2(i theta) = (e^{i theta} - 1 - i theta)/(i theta)^2
                     = (1 - cos(theta))/theta^2 + i (theta - sin(theta))/theta^2; series for |theta|<1 (R7)."""
    theta = np.asarray(theta, dtype=float)
    small = np.abs(theta) < 1.0
    th = np.where(small, 1.0, theta)
    big = (2.0 * np.sin(0.5 * th) ** 2) / th ** 2 + 1j * (th - np.sin(th)) / th ** 2
    ser = np.zeros(theta.shape, dtype=complex)
    z = 1j * np.where(small, theta, 0.0)
    for m in range(21, -1, -1):
        ser = ser * z + 1.0 / _FACT[m + 2]
    return np.where(small, ser, big)


def qr_mgs2(A, w, stats=None):
    """QR with respect to the weighted inner product <a,b> = w a^T b (Ensign gram_schmidt,
    PAPER.md:286, Fig. 1 line 22), modified Gram-Schmidt applied twice (R12).
    Returns basis Q (w Q^T Q = I) and coefficient R (upper triangular, R_jj > 0) with Q R = A."""
    N, r = A.shape
    sw = math.sqrt(w)
    Q = np.zeros((N, r))
    R = np.zeros((r, r))
    normA = math.sqrt(np.sum(A * A))
    for j in range(r):
        v = A[:, j].copy()
        for _pass in range(2):
            for i in range(j):
                c = Q[:, i] @ v
                v -= c * Q[:, i]
                R[i, j] += c
        nv = math.sqrt(v @ v)
        if nv <= 1e-14 * normA:               # rank-deficiency guard (R12), deterministic replacement
            if stats is not None:
                stats["qr_fallbacks"] = stats.get("qr_fallbacks", 0) + 1
            v = np.cos(2.0 * math.pi * (j + 1) * (np.arange(N) + 0.5) / N)
            for _pass in range(2):
                for i in range(j):
                    v -= (Q[:, i] @ v) * Q[:, i]
            Q[:, j] = v / math.sqrt(v @ v)
            R[j, j] = 0.0
        else:
            Q[:, j] = v / nv
            R[j, j] = nv
    return Q / sw, R * sw


# --------------------------------------------------------------------------------------
# flows of section 4
# --------------------------------------------------------------------------------------
def subflow_exact(Ah, Msym, t, s, g, d):
    """Exact solution of eq. (14)/(15) [(17)/(18) after diagonalisation], PAPER.md:246-264:
    Msym = T Lam T^T;  Ahat[k,:] <- (Ahat[k,:] T) o exp(s i t kt_d lam_j) T^T.
    s = -1 for the K equation (9) (term -d_x K C1^T), s = +1 for the L equation (11) (+d_v L D1^T)."""
    lam, T = jacobi_eigh(Msym)
    Mh = np.einsum("c...,cj->j...", Ah, T)
    ph = np.exp(s * 1j * t * g.kt(d)[None] * lam[:, None, None, None])
    return np.einsum("j...,cj->c...", ph * Mh, T)


def third_subflow(Ah, Msym, t, s, g, nonlin, order):
    """Eq. (16)/(19): d/dt Mhat = z/t Mhat + F(N(A)) T, z = s i t kt_3 lam_j,
    integrated by the exponential Euler method (order 1) or by the two-stage exponential
    Runge-Kutta method ETD2RK, c2 = 1 (order 2, reading R8; "a first or second order exponential
    Runge-Kutta method").  nonlin(Ag) evaluates N in real space."""
    lam, T = jacobi_eigh(Msym)
    theta = s * t * g.kt(2)[None] * lam[:, None, None, None]          # z = i theta
    ez = np.exp(1j * theta)
    Mh = np.einsum("c...,cj->j...", Ah, T)
    A0 = ifft3(Ah).real
    G0 = np.einsum("c...,cj->j...", fft3(nonlin(A0)), T)
    a = ez * Mh + t * phi1_imag(theta) * G0
    if order == 1:
        Mh_new = a
    else:
        Aa = ifft3(np.einsum("j...,cj->c...", a, T)).real
        G1 = np.einsum("c...,cj->j...", fft3(nonlin(Aa)), T)
        Mh_new = a + t * phi2_imag(theta) * (G1 - G0)
    return np.einsum("j...,cj->c...", Mh_new, T)


def _flow(A, t, g, Msym, s, nonlin, order):
    """K- or L-flow of length t: Lie-Trotter 1,2,3 (order 1) or classical Strang
    1(t/2),2(t/2),3(t),2(t/2),1(t/2) (order 2) of the directional sub-flows (R10)."""
    Ah = fft3(to_grid(A, g))
    if order == 1:
        Ah = subflow_exact(Ah, Msym[0], t, s, g, 0)
        Ah = subflow_exact(Ah, Msym[1], t, s, g, 1)
        Ah = third_subflow(Ah, Msym[2], t, s, g, nonlin, 1)
    else:
        Ah = subflow_exact(Ah, Msym[0], 0.5 * t, s, g, 0)
        Ah = subflow_exact(Ah, Msym[1], 0.5 * t, s, g, 1)
        Ah = third_subflow(Ah, Msym[2], t, s, g, nonlin, 2)
        Ah = subflow_exact(Ah, Msym[1], 0.5 * t, s, g, 1)
        Ah = subflow_exact(Ah, Msym[0], 0.5 * t, s, g, 0)
    return to_mat(ifft3(Ah).real)


def K_flow(K, t, C1, C2, E, gx, order):
    """Eq. (9): dK/dt = -sum_i d_{x_i}K C1_i^T + sum_i diag(E_i) K C2_i^T, E frozen."""
    def nonlin(Ag):
        Am = to_mat(Ag)
        out = np.zeros_like(Am)
        for d in range(3):
            out += E[d][:, None] * (Am @ C2[d].T)
        return to_grid(out, gx)
    return _flow(K, t, gx, [C1[d].T for d in range(3)], -1.0, nonlin, order)


def L_flow(L, t, D1, D2, gv, order):
    """Eq. (11): dL/dt = sum_i d_{v_i}L D1_i^T - sum_i diag(v_i) L D2_i^T (R9)."""
    vs = [gv.coord_flat(d) for d in range(3)]

    def nonlin(Ag):
        Am = to_mat(Ag)
        out = np.zeros_like(Am)
        for d in range(3):
            out -= vs[d][:, None] * (Am @ D2[d].T)
        return to_grid(out, gv)
    return _flow(L, t, gv, [D1[d].T for d in range(3)], +1.0, nonlin, order)


def S_flow(S, t, C1, C2, D1, D2):
    """Eq. (10): dS/dt = sum_i D2_i S C1_i^T - sum_i D1_i S C2_i^T, one classical RK4
    step of size t (R11)."""
    def rhs(Sm):
        out = np.zeros_like(Sm)
        for d in range(3):
            out += D2[d] @ Sm @ C1[d].T - D1[d] @ Sm @ C2[d].T
        return out
    k1 = rhs(S)
    k2 = rhs(S + 0.5 * t * k1)
    k3 = rhs(S + 0.5 * t * k2)
    k4 = rhs(S + t * k3)
    return S + (t / 6.0) * (k1 + 2.0 * k2 + 2.0 * k3 + k4)


# --------------------------------------------------------------------------------------
# Algorithms 1 and 2
# --------------------------------------------------------------------------------------
def step_alg1(X, S, V, tau, gx, gv, e_scale=1.0, stats=None, upto9=False):
    """Algorithm 1.  With upto9=True returns after line 9 (X1, L1, E0), which is
    what Algorithm 2 line 1 uses."""
    C1, C2, rho_t = coeff_C(V, gv)                         # line 1
    K0 = X @ S                                             # line 2
    E0 = field(K0, rho_t, gx, e_scale)                     # line 3, eq. (12)
    K1 = K_flow(K0, tau, C1, C2, E0, gx, 1)                # line 4
    X1, S1 = qr_mgs2(K1, gx.w, stats)                      # line 5
    D1, D2 = coeff_D(X1, E0, gx)                           # line 6
    S2 = S_flow(S1, tau, C1, C2, D1, D2)                   # line 7
    L0 = V @ S2.T                                          # line 8, L = V S^T
    L1 = L_flow(L0, tau, D1, D2, gv, 1)                    # line 9
    if upto9:
        return X1, L1, E0
    V1, R = qr_mgs2(L1, gv.w, stats)                       # line 10; S3 = R^T (Fig. 1 line 40)
    return X1, R.T.copy(), V1


def step_alg2(X, S, V, tau, gx, gv, e_scale=1.0, stats=None):
    """Algorithm 2."""
    X1, L1, _E0 = step_alg1(X, S, V, 0.5 * tau, gx, gv, e_scale, stats, upto9=True)   # line 1 (R13)
    Ehalf = field(X1, L1.T @ (gv.w * np.ones(gv.N)), gx, e_scale)    # line 2, eq. (13)
    C1, C2, _ = coeff_C(V, gv)                              # coefficients of V0 (as in line 1)
    K0 = X @ S
    K2 = K_flow(K0, 0.5 * tau, C1, C2, Ehalf, gx, 2)       # line 3
    X2, S3 = qr_mgs2(K2, gx.w, stats)                      # line 4
    D1, D2 = coeff_D(X2, Ehalf, gx)                        # line 5
    S4 = S_flow(S3, 0.5 * tau, C1, C2, D1, D2)             # line 6
    L = V @ S4.T                                           # line 7
    L2 = L_flow(L, tau, D1, D2, gv, 2)                     # line 8
    V1, R = qr_mgs2(L2, gv.w, stats)                       # line 9
    S5 = R.T.copy()
    C1, C2, _ = coeff_C(V1, gv)                            # line 10
    S6 = S_flow(S5, 0.5 * tau, C1, C2, D1, D2)             # line 11
    K3 = X2 @ S6                                           # line 12
    K4 = K_flow(K3, 0.5 * tau, C1, C2, Ehalf, gx, 2)       # line 13
    X3, S7 = qr_mgs2(K4, gx.w, stats)                      # line 14
    return X3, S7, V1

# --------------------------------------------------------------------------------------
# The unconventional ("BUG") integrator
# --------------------------------------------------------------------------------------
def S_flow_forward(S, t, C1, C2, D1, D2):
    """Galerkin S step of the unconventional integrator: the S equation is integrated FORWARD in time,
    dS/dt = X^T F(X S V^T) V = -(sum_i D2_i S C1_i^T - sum_i D1_i S C2_i^T)  (eq. (10), is the same
    right-hand side with the sign of the backward sub-flow (4)); one classical RK4 step (R11)."""
    def rhs(Sm):
        out = np.zeros_like(Sm)
        for d in range(3):
            out -= D2[d] @ Sm @ C1[d].T - D1[d] @ Sm @ C2[d].T
        return out
    k1 = rhs(S)
    k2 = rhs(S + 0.5 * t * k1)
    k3 = rhs(S + 0.5 * t * k2)
    k4 = rhs(S + t * k3)
    return S + (t / 6.0) * (k1 + 2.0 * k2 + 2.0 * k3 + k4)


def step_bug(X, S, V, tau, gx, gv, e_scale=1.0, stats=None):
    """One step of the unconventional (basis update & Galerkin) integrator, the paper's reference [4] (Ceruti &
    Lubich), which the paper names as supported by its framework but does not write out;
    restated here with the paper's sub-steps.  From (X0, S0, V0):
      K step: K(t0) = X0 S0, eq. (9) with the coefficients of V0 over tau -> QR -> X1 (R discarded), M = <X1, X0>;
      L step: L(t0) = V0 S0^T, eq. (11) with the coefficients of X0 over tau -> QR -> V1, N = <V1, V0>
              (both start from the SAME initial data: they are independent, unlike in Algorithm 1);
      S step: S(t0) = M S0 N^T, integrated forward with the coefficients of the NEW bases X1, V1 (S_flow_forward).
    Readings (the paper is silent, R19): first order, so E is frozen at E0 of eq. (12) for all three sub-steps
    (as Algorithm 1 does), the K and L flows are the Lie / exponential-Euler flows of Algorithm 1 (R13),
    <.,.> are the h^3-weighted inner products of Fig. 2.
    Returns (X1, S1, V1)."""
    C1, C2, rho_t = coeff_C(V, gv)
    K0 = X @ S
    E0 = field(K0, rho_t, gx, e_scale)                     # eq. (12)
    K1 = K_flow(K0, tau, C1, C2, E0, gx, 1)
    X1, _ = qr_mgs2(K1, gx.w, stats)
    M = gx.w * (X1.T @ X)
    D1, D2 = coeff_D(X, E0, gx)                            # coefficients of the OLD basis X0
    L0 = V @ S.T
    L1 = L_flow(L0, tau, D1, D2, gv, 1)
    V1, _ = qr_mgs2(L1, gv.w, stats)
    N = gv.w * (V1.T @ V)
    St = M @ S @ N.T
    C1n, C2n, _ = coeff_C(V1, gv)
    D1n, D2n = coeff_D(X1, E0, gx)
    S1 = S_flow_forward(St, tau, C1n, C2n, D1n, D2n)
    return X1, S1, V1


# --------------------------------------------------------------------------------------
# diagnostics (the quantities plotted in Figs. 4-7; definitions: R14)
# --------------------------------------------------------------------------------------
def moments(X, S, V, gx, gv, e_scale=1.0):
    ox = gx.w * X.sum(axis=0)                               # h_x^3 1^T X
    ov = gv.w * V.sum(axis=0)                               # h_v^3 V^T 1
    out = {"mass": float(ox @ S @ ov)}
    vs = [gv.coord_flat(d) for d in range(3)]
    out["momentum"] = [float(ox @ S @ (gv.w * (V.T @ vs[d]))) for d in range(3)]
    v2 = vs[0] ** 2 + vs[1] ** 2 + vs[2] ** 2
    out["kinetic_energy"] = float(0.5 * ox @ S @ (gv.w * (V.T @ v2)))
    E = field(X @ S, ov, gx, e_scale)                       # eq. (12) on the current factors
    out["electric_energy"] = float(0.5 * gx.w * np.sum(E * E))
    out["s_fro"] = float(math.sqrt(np.sum(S * S)))
    return out


def f_at(X, S, V, ix, iv):
    """f(x_p, v_p) = X[ix,:] S V[iv,:]^T  (rows of F = X S V^T)"""
    return np.einsum("pi,ij,pj->p", X[ix, :], S, V[iv, :])


def run(X, S, V, tau, nsteps, gx, gv, order=2, e_scale=1.0, probes=None):
    """advance nsteps steps; returns final factors and the history of the diagnostics"""
    stats = {}
    hist = [moments(X, S, V, gx, gv, e_scale)]
    for _ in range(nsteps):
        if order == 2:
            X, S, V = step_alg2(X, S, V, tau, gx, gv, e_scale, stats)
        elif order == "bug":
            X, S, V = step_bug(X, S, V, tau, gx, gv, e_scale, stats)
        else:
            X, S, V = step_alg1(X, S, V, tau, gx, gv, e_scale, stats)
        hist.append(moments(X, S, V, gx, gv, e_scale))
    fp = None if probes is None else f_at(X, S, V, probes[0], probes[1])
    return X, S, V, hist, fp, stats
