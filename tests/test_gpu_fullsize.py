"""Parity at BASELINE.json's full size, in the launch configuration bench.py times (configs[3]: 32^3 x 96, L5 = 12,
12-real links): the CUDA Mpc / Mpc^dagger in fp64, fp32 and 16-bit storage against the oracle evaluated one by
one on sampled odd sites (corners, all four wrap-arounds incl. the antiperiodic t boundary, and random sites).
Tolerances: north_star's 1e-12 / 1e-5; 2e-4 for the 16-bit operator."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

TOL = {"fp64": 1e-12, "fp32": 1e-5, "half": 2e-4}


def sample_sites(orc, n_random, seed):
    Lx, Ly, Lz, Lt = orc.L
    pts = []
    for t in (0, 1, Lt // 2, Lt - 2, Lt - 1):
        for z in (0, Lz - 1):
            for y in (0, Ly - 1):
                for x in (0, 1, Lx - 2, Lx - 1):
                    if (x + y + z + t) & 1:
                        pts.append(x + Lx * (y + Ly * (z + Lz * t)))
    rng = np.random.default_rng(seed)
    pts.extend(rng.choice(orc.sites_odd, size=n_random, replace=False).tolist())
    return np.unique(np.asarray(pts, dtype=np.int64))


def test_mpc_sampled_sites_at_config4():
    from conftest import rel
    from oracle.mdwf_oracle import MdwfOracle
    from paper_1701_07559_b200 import binding, inputs
    cfg = inputs.CONFIGS[3]
    L, L5 = cfg["L"], cfg["L5"]
    U = inputs.gauge_field(L, cfg["eps"], cfg["seed"], device="cuda")
    m = binding.Mdwf(L, L5, cfg["M5"], cfg["b5"], cfg["c5"], cfg["mf"])
    m.set_option("reconstruct", cfg["reconstruct"])
    m.load_gauge(U)
    orc = MdwfOracle(L, L5, cfg["M5"], cfg["b5"], cfg["c5"], cfg["mf"], U.cpu().numpy())
    del U
    b = inputs.gaussian_source(L, L5, cfg["seed"], device="cuda")
    V4 = L[0] * L[1] * L[2] * L[3]
    odd = torch.from_numpy(orc.sites_odd).cuda()
    bo_dev = b.reshape(L5, V4, 4, 3)[:, odd].contiguous()            # canonical parity layout [s][cb][4][3]
    b_host = b.cpu().numpy()
    del b
    torch.cuda.empty_cache()
    v_o = orc.parity_part(b_host, 1)
    del b_host
    sites = sample_sites(orc, 48, 7)
    cbs = torch.from_numpy(sites // 2).cuda()
    ref = {binding.OP_MPC: orc.Mpc_at_sites(v_o, sites), binding.OP_MPCDAG: orc.Mpc_at_sites(v_o, sites, dagger=True)}
    # auto = what bench.py times: the tile-sweep kernels (hop5_kernels.cuh) for fp32 storage at this size, hop3_kernels.cuh for
    # K1 and for 16-bit storage, hop_kernels.cuh for fp64; v3 = hop3_kernels.cuh for every fp32 kernel
    for kern, prec in (("auto", "fp64"), ("auto", "fp32"), ("auto", "half"), ("v3", "fp32")):
        m.set_option("kernels", kern)
        m.set_option("apply_precision", prec)
        x = bo_dev if prec == "fp64" else bo_dev.to(torch.complex64)
        for op, r in ref.items():
            got = m.apply(op, x)[:, cbs].cpu().numpy().astype(np.complex128)
            assert got.shape == r.shape
            assert rel(got, r) < TOL[prec], (kern, prec, op, rel(got, r))
            # every sampled site individually (a wrong wrap or sign shows up as an O(1) error on one site)
            per_site = np.linalg.norm((got - r).reshape(L5, len(sites), -1), axis=(0, 2)) / \
                np.linalg.norm(r.reshape(L5, len(sites), -1), axis=(0, 2))
            assert per_site.max() < 20 * TOL[prec], (prec, op, per_site.max())
    m.close()
