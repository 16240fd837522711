"""GPU parity for the full 4-step solve: mspcg_prepare_source (eq. 6, eq. 9),
mspcg_reconstruct_odd and mspcg_apply_full (eq. 4) against the numpy oracle, element by element, and the end-to-end
property: prepare -> mspcg_solve (CG and MSPCG) -> reconstruct -> the 2x2 operator of eq. (4) returns the source.

Tolerance: operator applications rel-L2 <= 1e-12 (fp64, BASELINE.json north_star).
"""
import numpy as np
import pytest

from oracle import Oracle
from paper_2104_05615_b200 import F16, F32, F64, Mspcg, synth

pytestmark = pytest.mark.gpu

MOB = dict(b=1.5, c=0.5, M5=1.8)


def rel(a, b):
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def setup(dims, Ls, mf, block, outer=F64, inner=F64, tb=-1, eps=0.3):
    import torch
    U = synth.gauge_natural_to_abi(synth.random_su3_links(dims, eps, 7), dims)
    ora = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf, block)
    ora.load_gauge(U, tb)
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf, block)
    g.configure(outer, inner, 18)
    g.load_gauge(U, tb)
    return ora, g, torch


def dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64).reshape(-1)).cuda()


# ragged tails of the 8/16/32-site tiles, an uncut direction, every compiled Ls, periodic and antiperiodic time
@pytest.mark.parametrize("dims,Ls,block,tb", [
    ((4, 4, 4, 4), 8, (2, 2, 2, 2), -1),
    ((2, 4, 6, 6), 4, (2, 2, 6, 2), -1),
    ((8, 4, 4, 6), 6, (4, 4, 2, 6), 1),
    ((4, 4, 4, 8), 12, (4, 2, 4, 4), -1),
    ((4, 6, 4, 4), 16, (2, 6, 2, 2), -1),
])
def test_prepare_reconstruct_full_vs_oracle(dims, Ls, block, tb):
    ora, g, torch = setup(dims, Ls, 0.03, block, tb=tb)
    phi_e = synth.gaussian_spinor_abi(dims, Ls, 41)
    phi_o = synth.gaussian_spinor_abi(dims, Ls, 42)
    psi_e = synth.gaussian_spinor_abi(dims, Ls, 43)
    want_hat, want_rhs = ora.prepare_source(phi_e, phi_o)
    hat, rhs = g.prepare_source(dev(torch, phi_e), dev(torch, phi_o))
    assert rel(hat.cpu().numpy(), want_hat) <= 1e-12
    assert rel(rhs.cpu().numpy(), want_rhs) <= 1e-12
    got = g.reconstruct_odd(dev(torch, psi_e), dev(torch, phi_o)).cpu().numpy()
    assert rel(got, ora.reconstruct_odd(psi_e, phi_o)) <= 1e-12
    oe, oo = g.apply_full(dev(torch, psi_e), dev(torch, phi_o))
    we, wo = ora.apply_full(psi_e, phi_o)
    assert rel(oe.cpu().numpy(), we) <= 1e-12 and rel(oo.cpu().numpy(), wo) <= 1e-12
    # parity really matters: an odd vector handed in as even gives something else
    he2, _ = g.prepare_source(dev(torch, phi_o), dev(torch, phi_e))
    assert rel(he2.cpu().numpy(), want_hat) > 1e-2
    g.close()


@pytest.mark.parametrize("use_precond,outer,inner", [(False, F64, F64), (True, F32, F16)])
def test_four_step_solve_returns_the_source(use_precond, outer, inner):
    """eq. (4) solved through eq. (5), (6), (9): apply_full(solution) == source, for plain CG in fp64 and for MSPCG with an
    fp32 sloppy outer iteration and the fp16 preconditioner."""
    dims, Ls, block = (8, 8, 8, 8), 8, (4, 4, 4, 4)
    ora, g, torch = setup(dims, Ls, 0.05, block, outer=outer, inner=inner, eps=0.25)
    phi_e = dev(torch, synth.gaussian_spinor_abi(dims, Ls, 51))
    phi_o = dev(torch, synth.gaussian_spinor_abi(dims, Ls, 52))
    hat, rhs = g.prepare_source(phi_e, phi_o)
    x, st = g.solve(rhs, tol=1e-11, max_iter=20000, use_precond=use_precond, n_inner=6, sloppy_prec=outer)
    assert st["converged"] and st["true_res"] <= 1e-10
    psi_o = g.reconstruct_odd(x, phi_o)
    oe, oo = g.apply_full(x, psi_o)
    assert float(torch.linalg.vector_norm(oo - phi_o) / torch.linalg.vector_norm(phi_o)) <= 1e-12   # exact by construction
    # |M psi - phi| is bounded by cond(D) times the normal-equation residual; the 8^4 test lattice gives < 1e-7
    assert float(torch.linalg.vector_norm(oe - phi_e) / torch.linalg.vector_norm(phi_e)) <= 1e-7
    g.close()


def test_errors():
    import torch
    dims, Ls = (4, 4, 4, 4), 8
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.01, (2, 2, 2, 2))
    g.configure(F64, F64, 18)
    v = dev(torch, synth.gaussian_spinor_abi(dims, Ls, 1))
    with pytest.raises(RuntimeError):
        g.prepare_source(v, v)        # no gauge field loaded
    g.close()
