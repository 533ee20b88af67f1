"""More oracle pins: P3 (link to the paper's Eq. (2)), P6 (dense brute force), P9 (CGLS invariants)."""
import numpy as np
import pytest

from conftest import gaussian, make_oracle, rel
from test_oracle_pins import DW_p, momentum, plane_wave


# ---- P3: the 5D operator reproduces the Moebius kernel of Eq. (2), PAPER.md:55-56 ------
@pytest.mark.parametrize("L5,M5,b5,c5,mf", [(8, 1.3, 1.5, 0.5, 0.05), (12, 1.3, 1.75, 0.75, 0.02),
                                            (6, 1.5, 1.3, 0.6, 0.1)])
def test_P3_overlap_identity_ties_D_to_eq2(L5, M5, b5, c5, mf):
    """(s=0,s'=0) block of P^+ D(1)^{-1} D(m_f) P  ==  (1+m)/2 + (1-m)/2 gamma5 eps_L5(gamma5 D^Moebius),
    D^Moebius = (b5+c5) D_W / (2 + (b5-c5) D_W)   [Eq. (2)],  eps_L(h) = ((1+h)^L-(1-h)^L)/((1+h)^L+(1-h)^L).
    D(m) is built column by column FROM THE ORACLE on plane waves (unit links)."""
    L = (4, 4, 2, 4)
    p = momentum(L, (1, 2, 1, 0))
    n = 4 * L5

    def dense_from_oracle(mass):
        orc = make_oracle(L, L5, M5, b5, c5, mass, 0.0, 0)
        M = np.zeros((n, n), complex)
        for j in range(n):
            chi = np.zeros((L5, 4, 3), complex)
            chi.reshape(n, 3)[j, 0] = 1.0
            out = orc.D(plane_wave(orc, p, chi))
            M[:, j] = out[:, 0, 0, 0, 0, :, 0].reshape(n)       # site x = 0, colour 0
        return M

    Dm, D1 = dense_from_oracle(mf), dense_from_oracle(1.0)
    Pp, Pm = np.diag([1.0, 1, 0, 0]), np.diag([0.0, 0, 1, 1])
    shift = np.roll(np.eye(L5), 1, axis=1)                      # (shift chi)_s = chi_{(s+1) mod L5}
    Pmat = np.kron(np.eye(L5), Pm) + np.kron(shift, Pp)
    K = Pmat.conj().T @ np.linalg.solve(D1, Dm) @ Pmat
    block = K[:4, :4]
    g5 = np.diag([1.0, 1, -1, -1])
    DW = DW_p(p, M5)
    Dmob = (b5 + c5) * DW @ np.linalg.inv(2 * np.eye(4) + (b5 - c5) * DW)        # Eq. (2)
    lam, V = np.linalg.eigh(g5 @ Dmob)
    assert np.allclose(g5 @ Dmob, (g5 @ Dmob).conj().T)
    eps_l = ((1 + lam) ** L5 - (1 - lam) ** L5) / ((1 + lam) ** L5 + (1 - lam) ** L5)     # eps_L5 on the eigenvalues
    eps = V @ np.diag(eps_l) @ V.conj().T
    Dov = 0.5 * (1 + mf) * np.eye(4) + 0.5 * (1 - mf) * g5 @ eps
    assert np.linalg.norm(block - Dov) / np.linalg.norm(Dov) < 1e-8


# ---- P6: dense brute force -----------------------------------------------------------------
@pytest.mark.parametrize("L,L5", [((2, 2, 2, 2), 4), ((4, 2, 2, 4), 3)])
def test_P6_dense_brute_force(L, L5):
    orc = make_oracle(L, L5, 1.3, 1.5, 0.5, 0.05, 0.5, 21)
    n = L5 * orc.V4 * 12
    Dd = np.zeros((n, n), complex)
    e = orc.zeros()
    ef = e.reshape(n)
    for j in range(n):
        ef[j] = 1.0
        Dd[:, j] = orc.D(e).reshape(n)
        ef[j] = 0.0
    idx = np.arange(n).reshape(L5, orc.V4, 12)
    ie, io = idx[:, orc.sites_even].ravel(), idx[:, orc.sites_odd].ravel()
    Dee, Deo, Doe, Doo = Dd[np.ix_(ie, ie)], Dd[np.ix_(ie, io)], Dd[np.ix_(io, ie)], Dd[np.ix_(io, io)]
    # D_ee = A on every site: compare with the oracle's A applied to unit vectors through a random probe
    v = gaussian(orc, 5)
    vf = v.reshape(n)
    assert rel(Dee @ vf[ie], orc.A(v, orc.sites_even).reshape(n)[ie]) < 1e-13
    assert rel(Doo @ vf[io], orc.A(v, orc.sites_odd).reshape(n)[io]) < 1e-13
    vo, ve = orc.parity_part(v, 1), orc.parity_part(v, 0)
    assert rel(Deo @ vf[io], orc.D_eo(vo).reshape(n)[ie]) < 1e-13
    assert rel(Doe @ vf[ie], orc.D_oe(ve).reshape(n)[io]) < 1e-13
    # Schur complement from the dense blocks == Mpc applied; its conjugate transpose == Mpcdag
    S = Doo - Doe @ np.linalg.solve(Dee, Deo)
    assert rel(orc.Mpc(vo).reshape(n)[io], S @ vf[io]) < 1e-12
    assert rel(orc.Mpcdag(vo).reshape(n)[io], S.conj().T @ vf[io]) < 1e-12
    assert np.abs(orc.Mpc(vo).reshape(n)[ie]).max() == 0.0
    # dense adjoint of D == Ddag
    assert rel(orc.Ddag(v).reshape(n), Dd.conj().T @ vf) < 1e-13
    # site-sampled evaluation agrees with the full one
    some = orc.sites_odd[[0, 3, len(orc.sites_odd) - 1]]
    full = orc.Mpc(vo).reshape(L5, orc.V4, 4, 3)[:, some]
    assert rel(orc.Mpc_at_sites(vo, some), full) < 1e-14
    fulld = orc.Mpcdag(vo).reshape(L5, orc.V4, 4, 3)[:, some]
    assert rel(orc.Mpc_at_sites(vo, some, dagger=True), fulld) < 1e-14
    # D8/D9: Schur solve with CGLS == dense solve
    b = gaussian(orc, 9)
    x_dense = np.linalg.solve(Dd, b.reshape(n))
    x, iters, res = orc.solve(b, tol=1e-12, maxiter=2000)
    assert res < 1e-11
    assert rel(x.reshape(n), x_dense) < 1e-10
    bp = orc.schur_prepare(b)
    assert rel(bp.reshape(n)[io], b.reshape(n)[io] - Doe @ np.linalg.solve(Dee, b.reshape(n)[ie])) < 1e-13
    # pack / unpack round trip and ordering: cb = lex/2 over odd sites
    pk = orc.pack_parity(v, 1)
    assert pk.shape == (L5, orc.V4 // 2, 4, 3)
    assert np.array_equal(orc.unpack_parity(pk, 1), vo)
    assert np.array_equal(orc.sites_odd // 2, np.arange(orc.V4 // 2))


# ---- P9: CGLS invariants on configs[0] -----------------------------------------------------
def test_P9_cgls_invariants(orc_cfg1):
    orc = orc_cfg1
    b = gaussian(orc, orc_cfg1_seed := 0)
    bp = orc.schur_prepare(b)
    bn = np.sqrt(orc.redot(bp, bp, orc.sites_odd))
    drift = []

    def cb(k, x, rho):
        if k % 10 == 0:
            true = bp - orc.Mpc(x)
            drift.append(np.linalg.norm((true - rho).ravel()) / bn)

    x_o, iters, hist = orc.cgls(bp, 1e-10, 1000, callback=cb)
    assert 10 < iters < 400                     # P10 sanity band: free-field estimate ~50
    assert all(h1 <= h0 * (1 + 1e-12) for h0, h1 in zip(hist, hist[1:]))   # ||rho_k|| non-increasing
    assert max(drift) < 1e-10
    x = orc.schur_reconstruct(b, x_o)
    assert orc.true_residual(b, x) < 1e-10
    # A7: ||b - D x|| equals ||b' - Mpc x_o|| when x_e is reconstructed exactly
    r_full = b - orc.D(x)
    r_pc = bp - orc.Mpc(x_o)
    assert abs(np.linalg.norm(r_full.ravel()) - np.linalg.norm(r_pc.ravel())) < 1e-9 * np.linalg.norm(r_pc.ravel()) + 1e-13
