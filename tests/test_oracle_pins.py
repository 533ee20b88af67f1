"""Pins of the CPU oracle against things OTHER than itself.

Nothing here needs a GPU.  Every expected value is a closed form, an invariant or a dense
numpy construction written in this file; none comes from the CUDA path.
"""
import numpy as np
import pytest

from conftest import gaussian, make_oracle, rel
from oracle import mdwf_oracle as mo

# ---- independent restatement of the algebra (numpy only) ------------------------------
I2 = np.eye(2)
SIG = [np.array([[0, 1], [1, 0]], complex), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]], complex)]


def degrand_rossi():
    """gamma_k = [[0, i sigma'_k], [-i sigma'_k, 0]]-type chiral basis written from SURVEY.md D2."""
    g1 = np.array([[0, 0, 0, 1j], [0, 0, 1j, 0], [0, -1j, 0, 0], [-1j, 0, 0, 0]])
    g2 = np.array([[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]], complex)
    g3 = np.array([[0, 0, 1j, 0], [0, 0, 0, -1j], [-1j, 0, 0, 0], [0, 1j, 0, 0]])
    g4 = np.array([[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]], complex)
    return [g1, g2, g3, g4]


def T_matrix(L5, mf):
    T = np.zeros((L5, L5))
    for s in range(1, L5):
        T[s, s - 1] = 1.0
    T[0, L5 - 1] = -mf
    return T


def Lambda_matrix(L5, mf):
    """Lambda = T (x) P+  +  T^T (x) P-   on the index (s, spin)."""
    Pp = np.diag([1.0, 1, 0, 0])
    Pm = np.diag([0.0, 0, 1, 1])
    T = T_matrix(L5, mf)
    return np.kron(T, Pp) + np.kron(T.T, Pm)


def DW_p(p, M5):
    g = degrand_rossi()
    out = (4 - M5 - sum(np.cos(p))) * np.eye(4, dtype=complex)
    for mu in range(4):
        out = out + 1j * np.sin(p[mu]) * g[mu]
    return out


def D5_p(p, L5, M5, b5, c5, mf):
    """dense 4L5 x 4L5 momentum-space operator D(p) = D_W(p) (b5 + c5 Lambda) + (1 - Lambda)."""
    Lam = Lambda_matrix(L5, mf)
    one = np.eye(4 * L5)
    return np.kron(np.eye(L5), DW_p(p, M5)) @ (b5 * one + c5 * Lam) + (one - Lam)


def plane_wave(orc, p, chi):
    """psi(x,s)[spin,colour] = exp(i p.x) chi[s,spin,colour]"""
    Lx, Ly, Lz, Lt = orc.L
    x = np.arange(Lx)[None, None, None, :]
    y = np.arange(Ly)[None, None, :, None]
    z = np.arange(Lz)[None, :, None, None]
    t = np.arange(Lt)[:, None, None, None]
    ph = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    return ph[None, ..., None, None] * chi[:, None, None, None, None, :, :]


def momentum(L, n):
    return np.array([2 * np.pi * n[0] / L[0], 2 * np.pi * n[1] / L[1], 2 * np.pi * n[2] / L[2],
                     2 * np.pi * (n[3] + 0.5) / L[3]])


# ---- gamma algebra (D2) ----------------------------------------------------------------
def test_gamma_basis():
    g = [mo.gamma(mu) for mu in range(5)]
    ref = degrand_rossi()
    for mu in range(4):
        assert np.array_equal(g[mu], ref[mu])
        assert np.allclose(g[mu], g[mu].conj().T)
        for nu in range(4):
            assert np.allclose(g[mu] @ g[nu] + g[nu] @ g[mu], 2 * np.eye(4) * (mu == nu))
    assert np.allclose(g[0] @ g[1] @ g[2] @ g[3], np.diag([1, 1, -1, -1]))
    assert np.array_equal(g[4], np.diag([1, 1, -1, -1]).astype(complex))


# ---- P1 / P2: plane waves on unit links ------------------------------------------------
@pytest.mark.parametrize("n", [(0, 0, 0, 0), (1, 0, 2, 1), (3, 1, 1, 5)])
def test_P1_plane_wave_closed_form(n):
    L, L5, M5, b5, c5, mf = (4, 2, 4, 6), 6, 1.3, 1.5, 0.5, 0.05
    orc = make_oracle(L, L5, M5, b5, c5, mf, 0.0, 0)          # eps = 0: unit links
    assert np.allclose(orc.U, np.eye(3))
    rng = np.random.default_rng(5)
    chi = rng.normal(size=(L5, 4, 3)) + 1j * rng.normal(size=(L5, 4, 3))
    p = momentum(L, n)
    psi = plane_wave(orc, p, chi)
    Dp = D5_p(p, L5, M5, b5, c5, mf)
    expect_chi = np.einsum("ab,bc->ac", Dp, chi.reshape(L5 * 4, 3)).reshape(L5, 4, 3)
    assert rel(orc.D(psi), plane_wave(orc, p, expect_chi)) < 1e-13
    # D^+ is the conjugate transpose of D(p)
    expect_dag = np.einsum("ab,bc->ac", Dp.conj().T, chi.reshape(L5 * 4, 3)).reshape(L5, 4, 3)
    assert rel(orc.Ddag(psi), plane_wave(orc, p, expect_dag)) < 1e-13
    # P2: D_W(p)^+ D_W(p) is the scalar (4 - M5 - sum cos)^2 + sum sin^2
    w = orc.DW(psi)
    scal = (4 - M5 - np.sum(np.cos(p))) ** 2 + np.sum(np.sin(p) ** 2)
    assert abs(np.vdot(w, w).real / np.vdot(psi, psi).real - scal) < 1e-12 * scal
    assert rel(w, plane_wave(orc, p, np.einsum("ab,sbc->sac", DW_p(p, M5), chi))) < 1e-13


def test_P1b_constant_abelian_links_shift_the_momentum():
    """U_mu(x) = diag(exp(i theta_mu,a)) (sum_a theta = 0): colour a sees momentum p + theta_a.
    Catches U <-> U^dagger and forward/backward mix-ups that unit links cannot see."""
    L, L5, M5, b5, c5, mf = (4, 4, 2, 4), 4, 1.1, 1.25, 0.25, 0.1
    orc = make_oracle(L, L5, M5, b5, c5, mf, 0.0, 0)
    theta = np.array([[0.3, -0.1, -0.2], [0.7, 0.2, -0.9], [-0.4, 0.5, -0.1], [0.15, 0.25, -0.4]])
    for mu in range(4):
        orc.U[..., mu, :, :] = np.diag(np.exp(1j * theta[mu]))
    rng = np.random.default_rng(6)
    chi = rng.normal(size=(L5, 4, 3)) + 1j * rng.normal(size=(L5, 4, 3))
    p = momentum(L, (1, 3, 1, 2))
    psi = plane_wave(orc, p, chi)
    expect = np.zeros_like(chi)
    for a in range(3):
        Dp = D5_p(p + theta[:, a], L5, M5, b5, c5, mf)
        expect[:, :, a] = (Dp @ chi[:, :, a].reshape(-1)).reshape(L5, 4)
    assert rel(orc.D(psi), plane_wave(orc, p, expect)) < 1e-13


# ---- P4: hermiticity statements -------------------------------
def _Gamma5(orc, v):
    """Gamma5 = gamma5 R5, R5: s -> L5-1-s."""
    w = v[::-1].copy()
    w[..., 2:, :] *= -1
    return w


def test_P4_adjoints_and_gamma5_hermiticity(orc_ragged):
    orc = orc_ragged
    x, y = gaussian(orc, 1), gaussian(orc, 2)
    # (iii) true adjoints of the separately coded daggers
    assert abs(np.vdot(x, orc.D(y)) - np.vdot(orc.Ddag(x), y)) < 1e-12 * abs(np.vdot(x, x))
    assert abs(np.vdot(x, orc.hop(y, orc.sites_all)) - np.vdot(orc.hop(x, orc.sites_all, dagger=True), y)) \
        < 1e-12 * abs(np.vdot(x, x))
    xo, yo = orc.parity_part(x, 1), orc.parity_part(y, 1)
    assert abs(np.vdot(xo, orc.Mpc(yo)) - np.vdot(orc.Mpcdag(xo), yo)) < 1e-12 * abs(np.vdot(xo, xo))
    for op in (orc.A, orc.B, orc.Ainv, orc.Lam):
        assert abs(np.vdot(x, op(y, orc.sites_all)) - np.vdot(op(x, orc.sites_all, dagger=True), y)) \
            < 1e-12 * abs(np.vdot(x, x))
    # gamma5 H gamma5 = H^+
    g5y = y.copy()
    g5y[..., 2:, :] *= -1
    hg = orc.hop(g5y, orc.sites_all)
    hg[..., 2:, :] *= -1
    assert rel(hg, orc.hop(y, orc.sites_all, dagger=True)) < 1e-13
    # Gamma5 A Gamma5 = A^+, Gamma5 B Gamma5 = B^+
    for op in (orc.A, orc.B):
        assert rel(_Gamma5(orc, op(_Gamma5(orc, y), orc.sites_all)), op(y, orc.sites_all, dagger=True)) < 1e-13
    # (ii) Gamma5 (D D_-) Gamma5 = (D D_-)^+ with D_- = c5 D_W - 1 slice-wise; as a bilinear identity:
    Dm = lambda v: orc.c5 * orc.DW(v) - v
    DmH = lambda v: orc.c5 * ((4 - orc.M5) * v - 0.5 * orc.hop(v, orc.sites_all, dagger=True)) - v
    lhs = _Gamma5(orc, orc.D(Dm(_Gamma5(orc, y))))
    rhs = DmH(orc.Ddag(y))
    assert rel(lhs, rhs) < 1e-12


def test_P4_literal_gamma5R5_hermiticity_at_c5_zero():
    orc = make_oracle((2, 4, 2, 4), 6, 1.4, 1.3, 0.0, 0.07, 0.5, 3)
    y = gaussian(orc, 4)
    assert rel(_Gamma5(orc, orc.D(_Gamma5(orc, y))), orc.Ddag(y)) < 1e-13


# ---- P5: gauge covariance ---------------------------------------------------------------
def test_P5_gauge_covariance(orc_ragged):
    from oracle.mdwf_oracle import MdwfOracle
    from paper_1701_07559_b200 import inputs
    orc = orc_ragged
    Lx, Ly, Lz, Lt = orc.L
    g = inputs.random_su3(99, orc.V4).numpy().reshape(Lt, Lz, Ly, Lx, 3, 3)
    Ug = np.empty_like(orc.U)
    for mu, ax in enumerate((3, 2, 1, 0)):              # axis of U[t][z][y][x] that direction mu moves along
        g_fwd = np.roll(g, -1, axis=ax)                  # g(x + mu)
        Ug[..., mu, :, :] = np.einsum("...ab,...bc,...dc->...ad", g, orc.U[..., mu, :, :], g_fwd.conj())
    orc_g = MdwfOracle(orc.L, orc.L5, orc.M5, orc.b5, orc.c5, orc.mf, Ug)
    psi = gaussian(orc, 8)
    rot = lambda v: np.einsum("tzyxab,stzyxib->stzyxia", g, v)
    assert rel(orc_g.D(rot(psi)), rot(orc.D(psi))) < 1e-13
    po = orc.parity_part(psi, 1)
    assert rel(orc_g.Mpc(rot(po)), rot(orc.Mpc(po))) < 1e-13
    assert rel(orc_g.Mpcdag(rot(po)), rot(orc.Mpcdag(po))) < 1e-13


# ---- P7: A^{-1} closed form vs numeric inverse -----------------------------------------
@pytest.mark.parametrize("L5,M5,b5,c5,mf", [(8, 1.3, 1.5, 0.5, 0.05), (12, 1.1, 1.5, 0.5, 0.005),
                                            (5, 1.7, 2.0, 0.3, 0.9), (24, 1.3, 2.25, 1.25, 0.00216)])
def test_P7_Ainv_closed_form(L5, M5, b5, c5, mf):
    alpha, beta = b5 * (4 - M5) + 1, c5 * (4 - M5) - 1
    Aplus = alpha * np.eye(L5) + beta * T_matrix(L5, mf)
    tab = mo.Ainv_plus_table(L5, alpha, beta, mf)
    assert np.max(np.abs(tab - np.linalg.inv(Aplus))) < 1e-14 * np.max(np.abs(tab)) * L5
    assert np.max(np.abs(tab.T - np.linalg.inv(Aplus.T))) < 1e-14 * np.max(np.abs(tab)) * L5


def test_P7_Ainv_applied(orc_ragged):
    orc = orc_ragged
    v = gaussian(orc, 3)
    for dag in (False, True):
        assert rel(orc.A(orc.Ainv(v, orc.sites_all, dag), orc.sites_all, dag), v) < 1e-14
        assert rel(orc.Ainv(orc.A(v, orc.sites_all, dag), orc.sites_all, dag), v) < 1e-14
    # against the dense (s,spin) matrix built here
    Amat = orc.alpha * np.eye(4 * orc.L5) + orc.beta * Lambda_matrix(orc.L5, orc.mf)
    vv = v.reshape(orc.L5, orc.V4, 4, 3)
    ref = np.einsum("SIsi,svic->SVIc".replace("V", "v"), np.linalg.inv(Amat).reshape(orc.L5, 4, orc.L5, 4), vv)
    assert rel(orc.Ainv(v, orc.sites_all).reshape(ref.shape), ref) < 1e-13
    refA = np.einsum("SIsi,svic->SvIc", Amat.reshape(orc.L5, 4, orc.L5, 4), vv)
    assert rel(orc.A(v, orc.sites_all).reshape(refA.shape), refA) < 1e-14


# ---- P8: special cases -------------------------------------------------------------------
def test_P8_shamir_limit_and_zero_links():
    L, L5, M5, mf = (2, 4, 4, 4), 6, 1.8, 0.04
    orc = make_oracle(L, L5, M5, 1.0, 0.0, mf, 0.3, 5)            # b5 = 1, c5 = 0: Shamir
    psi = gaussian(orc, 1)
    up = np.roll(psi, 1, axis=0)                                   # psi_{s-1}
    up[0] *= -mf
    dn = np.roll(psi, -1, axis=0)                                  # psi_{s+1}
    dn[-1] *= -mf
    shamir = orc.DW(psi) + psi
    shamir[..., :2, :] -= up[..., :2, :]                           # - P+ psi_{s-1}
    shamir[..., 2:, :] -= dn[..., 2:, :]                           # - P- psi_{s+1}
    assert rel(orc.D(psi), shamir) < 1e-14
    # links set to zero: H = 0 and D = A
    orc2 = make_oracle(L, L5, M5, 1.5, 0.5, mf, 0.3, 5)
    orc2.U[:] = 0
    Amat = orc2.alpha * np.eye(4 * L5) + orc2.beta * Lambda_matrix(L5, mf)
    ref = np.einsum("SIsi,svic->SvIc", Amat.reshape(L5, 4, L5, 4), psi.reshape(L5, orc2.V4, 4, 3))
    assert rel(orc2.D(psi).reshape(ref.shape), ref) < 1e-14
