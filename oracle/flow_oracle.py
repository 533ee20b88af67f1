"""CPU oracle for the gradient-flow smearing of the gauge field.  TEST INFRASTRUCTURE ONLY.

Only tests/ may import this module; it never imports paper_1701_07559_b200 and the CUDA path never imports it.

What the paper says: Sec. III smears the HISQ gauge fields with the gradient flow, "an infinitesimal
stout-smearing procedure [130]", to a flow time t_gf = 1.0; App. D solves "the
gradient flow equations with the Symanzik action ... with a step size of eps = 0.03 and up to n = 166 iterations".  The flow
equation and the integrator are in the cited literature ([127-130], Luescher), not in the paper.  Readings (N4-N6):

  F1  Flow equation   dV_mu(x)/dt = Z_mu(x)[V] V_mu(x),   Z = -g0^2 d_{x,mu} S(V)  (Lie-algebra valued),  V(0) = U.
  F2  Action          S = (2/g0^2) [ c0 sum_{x, mu<nu} Re tr(1 - P_{mu nu}(x)) + c1 sum_{x, mu != nu} Re tr(1 - R_{mu nu}(x)) ],
                      P the 1x1 plaquette, R_{mu nu} the 2x1 rectangle with its long side along mu.
                      Wilson flow (infinitesimal stout smearing, Sec. III): c0 = 1, c1 = 0.
                      Symanzik flow (App. D): tree-level Luescher-Weisz c0 = 5/3, c1 = -1/12.
                      With these normalisations  Z_mu(x) = -TA( V_mu(x) A_mu(x) ),  A = c0 (6 plaquette staples) + c1 (18
                      rectangle staples),  TA(M) = (M - M^+)/2 - tr(M - M^+)/6.
  F3  Integrator      Luescher's third-order Runge-Kutta, step eps:  Z_i = eps Z(W_i),
                      W1 = exp(Z0/4) W0,  W2 = exp(8/9 Z1 - 17/36 Z0) W1,  V(t+eps) = exp(3/4 Z2 - 8/9 Z1 + 17/36 Z0) W2.
  F4  Boundaries      periodic in all four directions (the antiperiodic time boundary belongs to the fermions).

Z is written out as -TA of the sum of every closed loop of F2 through the link (2 plaquettes and 6 rectangles per
transverse direction, each spelled out link by link), the action as plain sums over plaquettes and rectangles;
tests/test_oracle_flow.py pins the one against finite differences of the other, and the whole against the closed-form
decay rate of an abelian plane wave (khat^2, khat^2 + khat^4/12), exact invariances and the order of the integrator.

Layout: U[t][z][y][x][mu][3][3] complex128, mu in (x, y, z, t); U_mu(x) is the link from x to x + mu.
"""
import numpy as np

AXIS = {0: 3, 1: 2, 2: 1, 3: 0}          # direction mu -> array axis of U[t][z][y][x]


def shift(F, mu, n=1):
    """F(x + n mu) as a field of x (periodic)."""
    return np.roll(F, -n, axis=AXIS[mu])


def mul(*Ms):
    out = Ms[0]
    for M in Ms[1:]:
        out = out @ M
    return out


def dag(M):
    return np.conj(np.swapaxes(M, -1, -2))


def plaquette_field(U, mu, nu):
    """P_{mu nu}(x) = U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+"""
    Um, Un = U[..., mu, :, :], U[..., nu, :, :]
    return mul(Um, shift(Un, mu), dag(shift(Um, nu)), dag(Un))


def rectangle_field(U, mu, nu):
    """R_{mu nu}(x) = U_mu(x) U_mu(x+mu) U_nu(x+2mu) U_mu(x+mu+nu)^+ U_mu(x+nu)^+ U_nu(x)^+   (2 x 1, long side mu)"""
    Um, Un = U[..., mu, :, :], U[..., nu, :, :]
    return mul(Um, shift(Um, mu), shift(Un, mu, 2), dag(shift(shift(Um, mu), nu)), dag(shift(Um, nu)), dag(Un))


def action(U, c0=1.0, c1=0.0):
    """g0^2 S of F2."""
    s = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            s += c0 * np.sum(3.0 - np.trace(plaquette_field(U, mu, nu), axis1=-2, axis2=-1).real)
    if c1 != 0.0:
        for mu in range(4):
            for nu in range(4):
                if nu != mu:
                    s += c1 * np.sum(3.0 - np.trace(rectangle_field(U, mu, nu), axis1=-2, axis2=-1).real)
    return 2.0 * s


def mean_plaquette(U):
    """<Re tr P> / 3 over the 6 planes."""
    s = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            s += np.mean(np.trace(plaquette_field(U, mu, nu), axis1=-2, axis2=-1).real)
    return s / 18.0


def TA(M):
    A = 0.5 * (M - dag(M))
    tr = np.trace(A, axis1=-2, axis2=-1) / 3.0
    return A - tr[..., None, None] * np.eye(3)


def loops_through_link(U, mu, c0, c1):
    """Sum over all closed loops of the action that contain the link (x, mu), each written as the ordered product that STARTS
    with U_mu(x) and is traversed in the link's direction:  L_mu(x) = sum_loops  w_loop  U_mu(x) (rest of the loop).
    Loops of F2 traversed against the link enter through their reverse (Re tr is the same).  Then
    g0^2 S = const - 2 sum_loops w Re tr(loop), so the Lie derivative at the link is  d/ds S(e^{sX} U) = -2 Re tr(X L)."""
    Um = U[..., mu, :, :]
    L = np.zeros_like(Um)
    for nu in range(4):
        if nu == mu:
            continue
        Un = U[..., nu, :, :]
        # plaquettes in the (mu, nu) plane: above and below the link
        L += c0 * plaquette_field(U, mu, nu)
        L += c0 * mul(Um, dag(shift(shift(Un, mu), nu, -1)), dag(shift(Um, nu, -1)), shift(Un, nu, -1))
        if c1 == 0.0:
            continue
        # rectangles with the long side along mu: the link is the first or the second of the two long-side links (above / below)
        L += c1 * rectangle_field(U, mu, nu)                                                      # first link, above
        L += c1 * mul(Um, shift(Un, mu), dag(shift(Um, nu)), dag(shift(shift(Um, mu, -1), nu)),   # second link, above
                      dag(shift(Un, mu, -1)), shift(Um, mu, -1))
        L += c1 * mul(Um, shift(Um, mu), dag(shift(shift(Un, mu, 2), nu, -1)), dag(shift(shift(Um, mu), nu, -1)),   # first link, below
                      dag(shift(Um, nu, -1)), shift(Un, nu, -1))
        L += c1 * mul(Um, dag(shift(shift(Un, mu), nu, -1)), dag(shift(Um, nu, -1)), dag(shift(shift(Um, mu, -1), nu, -1)),   # second, below
                      shift(shift(Un, mu, -1), nu, -1), shift(Um, mu, -1))
        # rectangles with the long side along nu (R_{nu mu}): the link is a short side, at the bottom or at the top
        L += c1 * mul(Um, shift(Un, mu), shift(shift(Un, mu), nu), dag(shift(Um, nu, 2)), dag(shift(Un, nu)), dag(Un))       # up by two
        L += c1 * mul(Um, dag(shift(shift(Un, mu), nu, -1)), dag(shift(shift(Un, mu), nu, -2)), dag(shift(Um, nu, -2)),      # down by two
                      shift(Un, nu, -2), shift(Un, nu, -1))
    return L


def Z_field(U, c0=1.0, c1=0.0):
    """Z_mu(x) of F1/F2 for every link: the Lie-algebra element with  d/ds g0^2 S(e^{sX} U at (x,mu)) = 2 tr(X Z)  for all X,
    i.e. Z = -TA(L) with L the sum of loops through the link."""
    Z = np.zeros_like(U)
    for mu in range(4):
        Z[..., mu, :, :] = -TA(loops_through_link(U, mu, c0, c1))
    return Z


def expm_ah(X):
    """exp of antihermitian 3x3 matrices through the eigendecomposition of the Hermitian -iX."""
    w, V = np.linalg.eigh(-1j * X)
    return (V * np.exp(1j * w)[..., None, :]) @ dag(V)


def rk3_step(U, eps, c0=1.0, c1=0.0):
    """one step of F3"""
    Z0 = eps * Z_field(U, c0, c1)
    W1 = expm_ah(0.25 * Z0) @ U
    Z1 = eps * Z_field(W1, c0, c1)
    W2 = expm_ah((8.0 / 9.0) * Z1 - (17.0 / 36.0) * Z0) @ W1
    Z2 = eps * Z_field(W2, c0, c1)
    return expm_ah(0.75 * Z2 - (8.0 / 9.0) * Z1 + (17.0 / 36.0) * Z0) @ W2


def flow(U, eps, nsteps, c0=1.0, c1=0.0):
    V = U.copy()
    for _ in range(nsteps):
        V = rk3_step(V, eps, c0, c1)
    return V


WILSON = (1.0, 0.0)
SYMANZIK = (5.0 / 3.0, -1.0 / 12.0)
