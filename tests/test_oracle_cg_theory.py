"""Pins for the OUTER solver of the oracle (Algorithm 1, with the Polak-Ribiere beta of
eq. 18) against what CG theory fixes.  CPU only.

Every pin here fails for a solver whose beta is wrong (a dropped term, a wrong sign, the numerator
<z_{k+1}, r_k> instead of <z_{k+1}, r_{k+1} - r_k>): such a loop degenerates to steepest descent, which still
converges to the right x, so "x equals the dense solve" pins nothing about the path.

 (i)   finite termination: on an SPD matrix with m distinct eigenvalues CG ends in m steps;
 (ii)  conjugacy <p_{k+1}, A p_k> = 0 and orthogonality <r_{k+1}, z_k> = 0 with a fixed linear SPD preconditioner;
 (iii) with a fixed linear M the Polak-Ribiere beta equals the Fletcher-Reeves beta <z',r'>/<z,r> of Alg. 1 to rounding,
       so the residual history equals that of the textbook loop written out below;
 (iv)  iteration counts within +-2 of that textbook loop, also on the MDWF operator for both oracles (numpy and C).
"""
import numpy as np

from oracle import Oracle, solvers
from oracle.cbind import OracleC
from paper_2104_05615_b200 import synth

MOB = dict(b=1.5, c=0.5, M5=1.8)


def textbook_pcg(A, b, Minv=None, tol=1e-10, max_iter=100000):
    """Algorithm 1 exactly as printed: Fletcher-Reeves beta, x0 = 0.  Returns x, |r_k|/|b| list."""
    x = np.zeros_like(b)
    r = b.copy()
    z = Minv(r) if Minv else r.copy()
    p = z.copy()
    rz = np.vdot(r, z).real
    bn = np.linalg.norm(b)
    hist = []
    for _ in range(max_iter):
        Ap = A(p)
        alpha = rz / np.vdot(p, Ap).real
        x = x + alpha * p
        r = r - alpha * Ap
        hist.append(np.linalg.norm(r) / bn)
        if hist[-1] <= tol:
            break
        z = Minv(r) if Minv else r.copy()
        rz_new = np.vdot(r, z).real
        p = z + (rz_new / rz) * p
        rz = rz_new
    return x, hist


def spd(n, eigs, seed):
    rng = np.random.default_rng(seed)
    Q, _ = np.linalg.qr(rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n)))
    return (Q * np.asarray(eigs)) @ Q.conj().T


def test_finite_termination_with_m_distinct_eigenvalues():
    n, m = 60, 5
    eigs = np.repeat([1.0, 3.0, 10.0, 40.0, 250.0], n // m)
    A = spd(n, eigs, 0)
    rng = np.random.default_rng(1)
    b = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    x, st = solvers.pcg(lambda v: A @ v, b, tol=1e-11)
    assert st["converged"] and st["iters"] <= m + 1, st
    assert np.linalg.norm(A @ x - b) <= 1e-10 * np.linalg.norm(b)


def test_iteration_count_and_history_match_textbook_cg_and_pcg():
    n = 200
    eigs = np.logspace(0, 2.5, n)                   # kappa = 316: late-iteration rounding does not separate equivalent recurrences yet
    A = spd(n, eigs, 2)
    rng = np.random.default_rng(3)
    b = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    _, h_ref = textbook_pcg(lambda v: A @ v, b, tol=1e-10)
    h = []
    _, st = solvers.pcg(lambda v: A @ v, b, tol=1e-10, history=h)
    assert st["converged"] and abs(st["iters"] - len(h_ref)) <= 2, (st["iters"], len(h_ref))
    assert np.allclose(h[:30], h_ref[:30], rtol=1e-6)     # equal recurrences; rounding separates the paths after ~40 steps
    # kappa = 1e4: mathematically equal recurrences drift apart in rounding after some hundred steps; a few per cent, not 100x
    A4 = spd(n, np.logspace(0, 4, n), 2)
    _, h4_ref = textbook_pcg(lambda v: A4 @ v, b, tol=1e-10)
    _, st4 = solvers.pcg(lambda v: A4 @ v, b, tol=1e-10)
    assert st4["converged"] and abs(st4["iters"] - len(h4_ref)) <= 0.05 * len(h4_ref), (st4["iters"], len(h4_ref))
    # (iii) fixed linear SPD preconditioner: PR == FR, so the textbook PCG path is reproduced
    Mi = spd(n, 1.0 / (eigs * (1 + 0.5 * np.sin(np.arange(n)))), 2)   # same eigenvectors, perturbed inverse spectrum
    _, hp_ref = textbook_pcg(lambda v: A @ v, b, lambda r: Mi @ r, tol=1e-10)
    hp = []
    _, stp = solvers.pcg(lambda v: A @ v, b, precond=lambda r: Mi @ r, tol=1e-10, history=hp)
    assert stp["converged"] and abs(stp["iters"] - len(hp_ref)) <= 2, (stp["iters"], len(hp_ref))
    assert len(hp_ref) < 0.2 * len(h_ref)            # the preconditioner is a good one; steepest descent would not show it
    n0 = min(10, len(hp_ref))
    assert np.allclose(hp[:n0], hp_ref[:n0], rtol=1e-6)


def test_conjugacy_of_search_directions_and_orthogonality():
    n = 80
    A = spd(n, np.logspace(0, 3, n), 4)
    Mi = spd(n, np.logspace(0, -2.5, n), 5)          # unrelated SPD preconditioner (different eigenvectors)
    rng = np.random.default_rng(6)
    b = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    ps, rs, zs = [], [], []

    def Aop(v):
        ps.append(v.copy())
        return A @ v

    def Mop(r):
        rs.append(r.copy())
        zs.append(Mi @ r)
        return zs[-1].copy()

    solvers.pcg(Aop, b, precond=Mop, tol=1e-30, max_iter=12)
    ps = ps[1:13]                                     # call 0 is r0 = b - A x0
    assert len(ps) == 12
    for k in range(len(ps) - 1):
        c = abs(np.vdot(ps[k + 1], A @ ps[k]))
        assert c <= 1e-9 * np.linalg.norm(ps[k + 1]) * np.linalg.norm(A @ ps[k]), (k, c)
    for k in range(len(rs) - 1):
        c = abs(np.vdot(rs[k + 1], zs[k]))
        assert c <= 1e-9 * np.linalg.norm(rs[k + 1]) * np.linalg.norm(zs[k]), (k, c)


def _pair(dims, Ls, mf, block, eps, seed=21):
    U = synth.gauge_natural_to_abi(synth.random_su3_links(dims, eps, seed), dims)
    a = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf, block)
    c = OracleC(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf, block)
    a.load_gauge(U, -1)
    c.load_gauge(U, -1)
    return a, c


def test_mdwf_cg_iterations_match_textbook_both_oracles():
    """(iv) on the MDWF operator: plain CG of both oracles within +-2 of the textbook loop, which needs 37 iterations here
    (the steepest-descent degeneration needs 119); MSPCG (nonlinear M) with eq. 18 within +-3 of the FR loop and below CG."""
    dims, Ls, block = (8, 4, 2, 2), 4, (4, 4, 2, 2)
    a, c = _pair(dims, Ls, 0.01, block, eps=0.25)
    b = synth.gaussian_spinor_abi(dims, Ls, 2)
    _, h_ref = textbook_pcg(lambda v: c.apply_MdagM(v), b, tol=1e-9)
    assert len(h_ref) <= 45
    _, sc = c.solve(b, tol=1e-9, nhist=len(h_ref))
    _, sa = a.solve(b, tol=1e-9)
    assert abs(sc["iters"] - len(h_ref)) <= 2 and abs(sa["iters"] - len(h_ref)) <= 2, (sc["iters"], sa["iters"], len(h_ref))
    n0 = min(len(h_ref), len(sc["history"])) - 2
    assert np.allclose(sc["history"][:n0], h_ref[:n0], rtol=1e-6)
    _, hp_ref = textbook_pcg(lambda v: c.apply_MdagM(v), b, lambda r: c.apply_precond(r, 6), tol=1e-9)
    _, scp = c.solve(b, tol=1e-9, use_precond=True, n_inner=6)
    _, sap = a.solve(b, tol=1e-9, use_precond=True, n_inner=6)
    assert abs(scp["iters"] - len(hp_ref)) <= 3 and abs(sap["iters"] - len(hp_ref)) <= 3, (scp["iters"], sap["iters"], len(hp_ref))
    assert scp["iters"] < 0.7 * sc["iters"]
