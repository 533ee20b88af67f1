"""Parity of the SURVEY.md 8(f) rows built so far against the oracle: NEXT-1 symmetric preconditioning (operators and
solve) and NEXT-3 4D <-> 5D maps.  Same tolerances as the hot path: 1e-12 (fp64), 1e-5 (fp32), solves to an
oracle-recomputed true residual <= 1e-10."""
import numpy as np
import pytest
import torch

from conftest import rel
from test_gpu_parity import CASES, TOL, setup, to_dev

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name", ["cfg1", "ragged", "l5_12", "lx32", "l5_24", "kappa1"])
@pytest.mark.parametrize("prec", ["fp64", "fp32", "half"])
def test_symmetric_operator_parity(name, prec):
    from paper_1701_07559_b200 import binding
    orc, m, b = setup(name, "12")
    m.set_option("apply_precision", prec)
    bo_full = orc.parity_part(b, 1)
    x = to_dev(orc.pack_parity(b, 1), prec)
    for op, r in ((binding.OP_MPC_SYM, orc.Mpc_sym(bo_full)), (binding.OP_MPCDAG_SYM, orc.Mpc_sym_dag(bo_full))):
        got = m.apply(op, x).cpu().numpy().astype(np.complex128)
        assert rel(got, orc.pack_parity(r, 1)) < TOL[prec], (name, prec, op)
    m.close()


@pytest.mark.parametrize("ladder", ["d", "ds", "dsh"])
@pytest.mark.parametrize("name", ["cfg1", "ragged"])
def test_symmetric_solve_true_residual_by_oracle(name, ladder):
    orc, m, b = setup(name)
    m.set_option("ladder", ladder)
    m.set_option("matpc", "sym")
    sol, iters, tr, rc = m.solve(torch.from_numpy(b).cuda(), tol=1e-10, maxiter=5000)
    res = orc.true_residual(b, sol.cpu().numpy())
    assert rc == 0 and res <= 1e-10, (rc, res, tr)
    if ladder == "d":
        x_ref, it_ref, _ = orc.solve_sym(b, tol=1e-10)
        assert rel(sol.cpu().numpy(), x_ref) < 1e-8
        assert abs(iters - it_ref) <= 3, (iters, it_ref)
    m.close()


@pytest.mark.parametrize("name", ["cfg1", "ragged", "l5_12"])
@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_wall_maps(name, prec):
    from paper_1701_07559_b200 import inputs
    orc, m, b = setup(name)
    L, L5 = CASES[name][0], CASES[name][1]
    eta = b[0] * 0.5 + b[L5 - 1]                                     # some 4D field [t][z][y][x][4][3]
    e = to_dev(eta, prec)
    tol = 1e-12 if prec == "fp64" else 1e-6
    got = m.wall_source(e).cpu().numpy().astype(np.complex128)
    assert np.array_equal(got, orc.wall_source(eta).astype(got.dtype)) or rel(got, orc.wall_source(eta)) < 1e-7
    got = m.wall_source(e, lift=True).cpu().numpy().astype(np.complex128)
    assert rel(got, orc.lift(eta)) < tol
    psi = to_dev(b, prec)
    for mid, ref in ((False, orc.wall_project(b)), (True, orc.midpoint(b))):
        got = m.wall_project(psi, midpoint=mid).cpu().numpy().astype(np.complex128)
        assert rel(got, ref) < 1e-7
    m.close()
