"""Pins of oracle/flow_oracle.py (gradient-flow smearing).

G1  Z is the Lie derivative of the action: for a random link and a random su(3) direction X, the central finite difference
    of g0^2 S(e^{sX} U) (the action coded as plain sums over plaquettes and rectangles) equals 2 tr(X Z).
G2  closed form: an abelian transverse plane wave of small amplitude decays as exp(-lambda t) with
    lambda = khat^2 (Wilson) and khat^2 + khat^4 / 12 (tree-level Symanzik), khat^2 = 4 sin^2(k/2): fixes the normalisation
    of the flow time (t_gf = 1 of PAPER.md:100 means smoothing radius sqrt(8 t)) and the rectangle weights.
G3  a pure gauge field is a fixed point; the flow commutes with gauge transformations.
G4  the integrator is third order: the one-step error falls by ~16 when eps is halved.
G5  the flow stays in SU(3), lowers the action monotonically and raises the mean plaquette.
"""
import numpy as np
import pytest

from oracle import flow_oracle as fo


def rand_su3_alg(rng, shape):
    G = rng.normal(size=shape + (3, 3)) + 1j * rng.normal(size=shape + (3, 3))
    return fo.TA(G)


def rand_field(rng, L, eps):
    Lx, Ly, Lz, Lt = L
    return fo.expm_ah(eps * rand_su3_alg(rng, (Lt, Lz, Ly, Lx, 4)))


@pytest.mark.parametrize("act", [fo.WILSON, fo.SYMANZIK])
def test_G1_force_is_the_derivative_of_the_action(act):
    rng = np.random.default_rng(1)
    L = (4, 4, 4, 6)
    U = rand_field(rng, L, 0.4)
    Z = fo.Z_field(U, *act)
    for trial in range(6):
        t, z, y, x, mu = (int(rng.integers(n)) for n in (L[3], L[2], L[1], L[0], 4))
        X = rand_su3_alg(rng, ())
        h = 1e-4
        vals = []
        for s in (+h, -h):
            V = U.copy()
            V[t, z, y, x, mu] = fo.expm_ah(s * X) @ U[t, z, y, x, mu]
            vals.append(fo.action(V, *act))
        fd = (vals[0] - vals[1]) / (2 * h)
        exact = 2.0 * np.trace(X @ Z[t, z, y, x, mu]).real
        assert abs(fd - exact) < 1e-6 * max(1.0, abs(exact)), (trial, fd, exact)
    assert np.max(np.abs(Z + fo.dag(Z))) < 1e-13 and np.max(np.abs(np.trace(Z, axis1=-2, axis2=-1))) < 1e-13


@pytest.mark.parametrize("act,lam", [(fo.WILSON, lambda k2: k2), (fo.SYMANZIK, lambda k2: k2 + k2 * k2 / 12.0)])
def test_G2_plane_wave_decay_rate(act, lam):
    L = (4, 8, 4, 4)
    Lx, Ly, Lz, Lt = L
    T = 1j * np.diag([0.5, -0.5, 0.0])                        # tr T^2 = -1/2
    n, a0 = 1, 1e-4
    k = 2 * np.pi * n / Ly
    theta = a0 * np.cos(k * np.arange(Ly))
    U = np.zeros((Lt, Lz, Ly, Lx, 4, 3, 3), complex)
    U[...] = np.eye(3)
    for y in range(Ly):
        U[:, :, y, :, 0] = fo.expm_ah(theta[y] * T)
    eps, nsteps = 0.02, 25
    V = fo.flow(U, eps, nsteps, *act)
    k2 = 4 * np.sin(k / 2) ** 2
    expect = np.exp(-lam(k2) * eps * nsteps)
    got = np.array([np.angle(V[0, 0, y, 0, 0, 0, 0]) * 2.0 for y in range(Ly)])      # U_00 = exp(i theta / 2)
    assert np.allclose(got, theta * expect, rtol=0, atol=2e-5 * a0)
    assert np.max(np.abs(V[..., 1:, :, :] - np.eye(3))) < 1e-12                        # the other directions stay trivial


def test_G3_pure_gauge_fixed_point_and_covariance():
    rng = np.random.default_rng(3)
    L = (4, 4, 4, 4)
    g = fo.expm_ah(rand_su3_alg(rng, (L[3], L[2], L[1], L[0])))
    Upg = np.stack([g @ fo.dag(fo.shift(g, mu)) for mu in range(4)], axis=4)
    for act in (fo.WILSON, fo.SYMANZIK):
        assert np.max(np.abs(fo.Z_field(Upg, *act))) < 1e-12
    U = rand_field(rng, L, 0.3)
    Ug = np.stack([g @ U[..., mu, :, :] @ fo.dag(fo.shift(g, mu)) for mu in range(4)], axis=4)
    V = fo.flow(U, 0.03, 2, *fo.SYMANZIK)
    Vg = fo.flow(Ug, 0.03, 2, *fo.SYMANZIK)
    ref = np.stack([g @ V[..., mu, :, :] @ fo.dag(fo.shift(g, mu)) for mu in range(4)], axis=4)
    assert np.max(np.abs(Vg - ref)) < 1e-12


def test_G4_third_order_integrator():
    rng = np.random.default_rng(4)
    U = rand_field(rng, (4, 4, 4, 4), 0.3)
    ref = fo.flow(U, 0.1 / 64, 64)
    e1 = np.linalg.norm(fo.flow(U, 0.1, 1) - ref)
    e2 = np.linalg.norm(fo.flow(U, 0.05, 2) - ref)
    assert e1 / e2 > 6.0 and e2 < e1, (e1, e2)                # global error O(eps^3): ratio ~ 8


def test_G5_smoothing():
    rng = np.random.default_rng(5)
    U = rand_field(rng, (4, 4, 4, 4), 0.5)
    for act in (fo.WILSON, fo.SYMANZIK):
        V, s_prev, p_prev = U, fo.action(U, *act), fo.mean_plaquette(U)
        for _ in range(5):
            V = fo.rk3_step(V, 0.03, *act)
            s, p = fo.action(V, *act), fo.mean_plaquette(V)
            assert s < s_prev and p > p_prev
            s_prev, p_prev = s, p
        assert np.max(np.abs(V @ fo.dag(V) - np.eye(3))) < 1e-13
        assert np.max(np.abs(np.linalg.det(V) - 1.0)) < 1e-13
