"""Parity of the SURVEY.md 8(f) rows built so far against the oracle: NEXT-1 symmetric preconditioning (operators and
solve) and NEXT-3 4D <-> 5D maps.  Same tolerances as the hot path: 1e-12 (fp64), 1e-5 (fp32), solves to an
oracle-recomputed true residual <= 1e-10."""
import numpy as np
import pytest
import torch

from conftest import rel
from test_gpu_parity import CASES, TOL, setup, to_dev

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name", ["cfg1", "ragged", "l5_12", "l5_16", "lx32", "l5_24", "kappa1", "tile16"])
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


@pytest.mark.parametrize("action", ["wilson", "symanzik"])
@pytest.mark.parametrize("L", [(4, 4, 4, 6), (6, 4, 2, 8), (2, 2, 4, 4)])
def test_gradient_flow_parity(action, L):
    """NEXT-4: the flowed links against the oracle, element by element (fp64), and the mean plaquette"""
    from oracle import flow_oracle as fo
    from paper_1701_07559_b200 import binding, inputs
    if min(L) < 4 and action == "symanzik":
        pytest.skip("2 x 1 rectangles wrap onto themselves on an extent of 2: the oracle's loop list assumes extents >= 3")
    U = inputs.gauge_field(L, 0.4, 31)
    m = binding.Mdwf(L, 8, 1.3, 1.5, 0.5, 0.05)
    Ud = U.cuda().contiguous()
    p0 = m.plaquette(Ud)
    assert abs(p0 - fo.mean_plaquette(U.numpy())) < 1e-13
    act = fo.WILSON if action == "wilson" else fo.SYMANZIK
    ref = fo.flow(U.numpy(), 0.03, 3, *act)
    p1 = m.gradient_flow(Ud, 0.03, 3, action)
    got = Ud.cpu().numpy()
    assert np.max(np.abs(got - ref)) < 1e-12
    assert abs(p1 - fo.mean_plaquette(ref)) < 1e-13 and p1 > p0
    m.close()


# ---- NEXT-2: batched (multi-right-hand-side) operator -----------------------------------------------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("name", ["cfg1", "l5_12", "l5_16", "lx32", "tile8"])
@pytest.mark.parametrize("prec", ["fp32", "half"])
def test_batched_operator_matches_single_and_oracle(name, prec):
    """mdwf_apply_batch on 5 right-hand sides: bit-identical to 5 single applications on the same (v3) kernels, and each against the
    oracle within the precision's tolerance"""
    from paper_1701_07559_b200 import binding, inputs
    from test_gpu_parity import setup, to_dev, rel, TOL
    orc, m, b = setup(name, "12")
    m.set_option("kernels", "v3")
    m.set_option("apply_precision", prec)
    nrhs = 5
    srcs = [b] + [inputs.gaussian_source(orc.L, orc.L5, 100 + r).numpy() for r in range(1, nrhs)]
    xs = torch.stack([to_dev(orc.pack_parity(s, 1), prec) for s in srcs]).contiguous()
    for op, ref in ((binding.OP_MPC, orc.Mpc), (binding.OP_MPCDAG, orc.Mpcdag)):
        got = m.apply_batch(op, xs)
        for r in range(nrhs):
            single = m.apply(op, xs[r].contiguous())
            assert torch.equal(got[r], single), (name, prec, op, r)
        for r in (0, nrhs - 1):
            want = orc.pack_parity(ref(orc.parity_part(srcs[r], 1)), 1)
            assert rel(got[r].cpu().numpy().astype(np.complex128), want) < TOL[prec], (name, prec, op, r)
    m.close()


@pytest.mark.gpu
def test_batched_operator_rejects_what_it_does_not_cover():
    from paper_1701_07559_b200 import binding
    from test_gpu_parity import setup, to_dev
    orc, m, b = setup("ragged")                      # L5 = 5: no batched kernel
    x = torch.stack([to_dev(orc.pack_parity(b, 1), "fp32")] * 2).contiguous()
    with pytest.raises(binding.MdwfError):
        m.apply_batch(binding.OP_MPC, x)
    with pytest.raises(binding.MdwfError):
        m.apply_batch(binding.OP_D, x)
    m.close()
