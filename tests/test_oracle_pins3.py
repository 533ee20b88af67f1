"""Pins of the oracle's SURVEY.md 8(f) functions (NEXT-1 symmetric preconditioning, NEXT-3 4D <-> 5D maps).

N1  lift / wall_project against the paper's Eq. (2) on an INTERACTING gauge field: with the dense
    4D overlap operator D_ov(m) = (1+m)/2 + (1-m)/2 gamma5 eps_L5(gamma5 D^Moebius) built from Eq. (2),
        D_ov(m)^{-1} eta = eta - (1 - m_f) q,   q = wall_project( D(m)^{-1} lift(eta) ).
    (Derivation: D(1) - D(m) = -(1-m) D_- W with W the wall injection, and P3's identity for D(1)^{-1} D(m).)
N2  wall_source / wall_project / midpoint against literal index loops.
N3  Mpc_sym against the dense Schur complement 1 - D_oo^{-1} D_oe D_ee^{-1} D_eo, its adjoint, and solve_sym = D^{-1} b.
"""
import numpy as np
import pytest

from conftest import gaussian, make_oracle, rel


def dense_D(orc):
    n = orc.L5 * orc.V4 * 12
    Dd = np.zeros((n, n), complex)
    e = orc.zeros()
    ef = e.reshape(n)
    for j in range(n):
        ef[j] = 1.0
        Dd[:, j] = orc.D(e).reshape(n)
        ef[j] = 0.0
    return Dd


def dense_DW4(orc):
    """the 4D Wilson kernel D_W(M5) of Eq. (2) as a dense matrix, read off slice 0 of the oracle's DW"""
    n4 = orc.V4 * 12
    M = np.zeros((n4, n4), complex)
    e = orc.zeros()
    for j in range(n4):
        e[0].reshape(n4)[j] = 1.0
        M[:, j] = orc.DW(e)[0].reshape(n4)
        e[0].reshape(n4)[j] = 0.0
    return M


@pytest.mark.parametrize("L5,M5,b5,c5,mf", [(4, 1.3, 1.5, 0.5, 0.05), (6, 1.2, 1.25, 0.25, 0.1)])
def test_N1_lift_solve_project_is_the_overlap_inverse_of_eq2(L5, M5, b5, c5, mf):
    orc = make_oracle((2, 2, 2, 2), L5, M5, b5, c5, mf, 0.4, 31)
    n4 = orc.V4 * 12
    DW = dense_DW4(orc)
    g5 = np.kron(np.eye(orc.V4), np.kron(np.diag([1.0, 1, -1, -1]), np.eye(3)))
    Dmob = (b5 + c5) * DW @ np.linalg.inv(2 * np.eye(n4) + (b5 - c5) * DW)          # Eq. (2)
    Hm = g5 @ Dmob
    assert np.allclose(Hm, Hm.conj().T, atol=1e-12)
    lam, V = np.linalg.eigh(Hm)
    eps_l = ((1 + lam) ** L5 - (1 - lam) ** L5) / ((1 + lam) ** L5 + (1 - lam) ** L5)
    Dov = 0.5 * (1 + mf) * np.eye(n4) + 0.5 * (1 - mf) * g5 @ (V @ np.diag(eps_l) @ V.conj().T)
    eta = gaussian(orc, 77)[0]                                                      # a 4D field [t][z][y][x][4][3]
    b5d = orc.lift(eta)
    psi = np.linalg.solve(dense_D(orc), b5d.reshape(-1)).reshape(orc.shape)
    q = orc.wall_project(psi)
    lhs = np.linalg.solve(Dov, eta.reshape(n4))
    rhs = (eta - (1.0 - mf) * q).reshape(n4)
    assert np.linalg.norm(lhs - rhs) / np.linalg.norm(lhs) < 1e-8
    # the oracle's own CG solve gives the same 4D answer
    x, iters, res = orc.solve(b5d, tol=1e-11, maxiter=4000)
    assert rel(orc.wall_project(x), q) < 1e-8


def test_N2_maps_by_literal_loops():
    orc = make_oracle((2, 2, 2, 4), 6, 1.3, 1.5, 0.5, 0.05, 0.3, 5)
    L5 = orc.L5
    eta = gaussian(orc, 3)[1]
    b = orc.wall_source(eta)
    psi = gaussian(orc, 4)
    q, Q = orc.wall_project(psi), orc.midpoint(psi)
    for sp in range(4):
        up = sp < 2                                    # gamma5 = diag(+,+,-,-): P+ keeps spins 0,1
        for s in range(L5):
            want = eta[..., sp, :] if ((s == 0 and up) or (s == L5 - 1 and not up)) else 0.0
            assert np.array_equal(b[s][..., sp, :], want + 0 * b[s][..., sp, :])
        assert np.array_equal(q[..., sp, :], psi[L5 - 1][..., sp, :] if up else psi[0][..., sp, :])
        assert np.array_equal(Q[..., sp, :], psi[L5 // 2 - 1][..., sp, :] if up else psi[L5 // 2][..., sp, :])
    # D_- = c5 D_W - 1 and D = D_+ + D_- Lambda with D_+ = b5 D_W + 1 (D6)
    v = gaussian(orc, 9)
    lam_v = orc.Lam(v, orc.sites_all)
    assert rel(orc.D(v), orc.b5 * orc.DW(v) + v + orc.Dminus(lam_v)) < 1e-13


@pytest.mark.parametrize("L,L5", [((2, 2, 2, 2), 4), ((4, 2, 2, 4), 3)])
def test_N3_symmetric_preconditioning_dense(L, L5):
    orc = make_oracle(L, L5, 1.3, 1.5, 0.5, 0.05, 0.5, 21)
    Dd = dense_D(orc)
    n = Dd.shape[0]
    idx = np.arange(n).reshape(L5, orc.V4, 12)
    ie, io = idx[:, orc.sites_even].ravel(), idx[:, orc.sites_odd].ravel()
    Dee, Deo, Doe, Doo = Dd[np.ix_(ie, ie)], Dd[np.ix_(ie, io)], Dd[np.ix_(io, ie)], Dd[np.ix_(io, io)]
    Msym = np.eye(len(io)) - np.linalg.solve(Doo, Doe @ np.linalg.solve(Dee, Deo))
    v = orc.parity_part(gaussian(orc, 5), 1)
    w = orc.parity_part(gaussian(orc, 6), 1)
    assert rel(orc.Mpc_sym(v).reshape(n)[io], Msym @ v.reshape(n)[io]) < 1e-12
    assert rel(orc.Mpc_sym_dag(v).reshape(n)[io], Msym.conj().T @ v.reshape(n)[io]) < 1e-12
    assert abs(np.vdot(w, orc.Mpc_sym(v)) - np.vdot(orc.Mpc_sym_dag(w), v)) < 1e-10 * abs(np.vdot(w, orc.Mpc_sym(v)))
    # Mpc_sym = A^{-1} Mpc
    assert rel(orc.Mpc_sym(v), orc.Ainv(orc.Mpc(v), orc.sites_odd)) < 1e-13
    b = gaussian(orc, 8)
    x, iters, res = orc.solve_sym(b, tol=1e-11, maxiter=4000)
    assert res <= 1e-11
    assert rel(x.reshape(n), np.linalg.solve(Dd, b.reshape(n))) < 1e-8
