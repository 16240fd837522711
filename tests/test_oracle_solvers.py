"""Pins for the oracle's block operator A_s, the multi-splitting preconditioner, CG and MSPCG.  CPU only."""
import numpy as np
import pytest

from oracle import Oracle, mdwf, solvers
from oracle.cbind import OracleC
from paper_2104_05615_b200 import synth

MOB = dict(b=1.5, c=0.5, M5=1.8)


def rel(a, b):
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b))


def pair(dims, Ls, mf, block, eps=0.35, seed=21, tb=-1):
    U = synth.gauge_natural_to_abi(synth.random_su3_links(dims, eps, seed), dims)
    a = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf, block)
    c = OracleC(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf, block)
    a.load_gauge(U, tb)
    c.load_gauge(U, tb)
    return a, c


def dense_of(apply, n):
    """Dense complex matrix of a (real-linear but complex-linear) operator on ABI vectors of n complex entries."""
    M = np.empty((n, n), dtype=np.complex128)
    e = np.zeros(2 * n)
    for j in range(n):
        e[:] = 0.0
        e[2 * j] = 1.0
        col = apply(e).reshape(-1)
        M[:, j] = col[0::2] + 1j * col[1::2]
    return M


def c2abi(z, shape):
    return np.stack([z.real, z.imag], axis=-1).reshape(shape)


def test_oracle_A_vs_B_cross_check():
    """Two independent restatements (numpy shifts vs C site loops) agree on every entry point."""
    dims, Ls, block = (4, 4, 2, 6), 2, (2, 4, 2, 2)
    a, c = pair(dims, Ls, 0.03, block)
    v = synth.gaussian_spinor_abi(dims, Ls, 5)
    assert rel(c.apply_MdagM(v), a.apply_MdagM(v)) < 1e-13
    assert rel(c.apply_D(v), a.apply_D(v)) < 1e-13
    assert rel(c.apply_D(v, True), a.apply_D(v, True)) < 1e-13
    for blk in (0, 3, c.num_blocks - 1):
        assert rel(c.apply_A_block(v, blk), a.apply_A_block(v, blk)) < 1e-13
    assert rel(c.apply_precond(v, 4), a.apply_precond(v, 4)) < 1e-11
    # same PCG path: residual histories of the first outer iterations agree (later ones drift by rounding, R18)
    ha = []
    a.solve(v, tol=1e-30, use_precond=True, n_inner=3, max_iter=6, history=ha)
    _, sc = c.solve(v, tol=1e-30, use_precond=True, n_inner=3, max_iter=6, nhist=6)
    assert np.allclose(ha, sc["history"], rtol=1e-8)
    ha = []
    a.solve(v, tol=1e-30, max_iter=10, history=ha)
    _, sc = c.solve(v, tol=1e-30, max_iter=10, nhist=10)
    assert np.allclose(ha, sc["history"], rtol=1e-9)


def test_dense_direct_solve_cg_and_mspcg():
    """north_star pin: dense-matrix direct solve vs CG and MSPCG on a tiny lattice (768 complex unknowns)."""
    dims, Ls, block = (4, 4, 2, 2), 4, (2, 2, 2, 2)
    a, c = pair(dims, Ls, 0.05, block)
    n = Ls * (int(np.prod(dims)) // 2) * 12
    A = dense_of(c.apply_MdagM, n)
    assert np.abs(A - A.conj().T).max() < 1e-12
    w = np.linalg.eigvalsh(A)
    assert w.min() > 0
    b = synth.gaussian_spinor_abi(dims, Ls, 7)
    bz = b.reshape(-1, 2)[:, 0] + 1j * b.reshape(-1, 2)[:, 1]
    x_direct = c2abi(np.linalg.solve(A, bz), b.shape)
    for orc in (a, c):
        x_cg, st = orc.solve(b, tol=1e-12)
        assert st["converged"] and rel(x_cg, x_direct) < 1e-10
        x_ms, st2 = orc.solve(b, tol=1e-12, use_precond=True, n_inner=4)
        assert st2["converged"] and rel(x_ms, x_direct) < 1e-10
        assert st2["iters"] < st["iters"]
    # the numpy dense D^dag D equals D^dag times D built separately
    Dm = dense_of(c.apply_D, n)
    assert np.abs(Dm.conj().T @ Dm - A).max() < 1e-12
    assert np.abs(dense_of(lambda v: c.apply_D(v, True), n) - Dm.conj().T).max() < 1e-12


def test_block_operator_dense_properties_and_exact_block_cg():
    """A_s (PAD) is Hermitian positive definite; k >= dim block CG reproduces A_s^-1 r_s; truncation differs."""
    dims, Ls, block = (4, 4, 2, 2), 2, (2, 2, 2, 2)
    a, c = pair(dims, Ls, 0.05, block)
    vh = int(np.prod(dims)) // 2
    n = Ls * vh * 12
    blk = 1
    As = dense_of(lambda v: c.apply_A_block(v, blk), n)
    sup = np.abs(As).sum(axis=0) > 0            # the block's interior degrees of freedom
    assert sup.sum() == Ls * 8 * 12
    assert np.abs(As[~sup]).max() == 0 and np.abs(As[:, ~sup]).max() == 0
    Ab = As[np.ix_(sup, sup)]
    assert np.abs(Ab - Ab.conj().T).max() < 1e-12
    assert np.linalg.eigvalsh(Ab).min() > 0
    r = synth.gaussian_spinor_abi(dims, Ls, 8)
    rz = (r.reshape(-1, 2)[:, 0] + 1j * r.reshape(-1, 2)[:, 1])
    want = np.zeros(n, dtype=np.complex128)
    want[sup] = np.linalg.solve(Ab, rz[sup])
    got = c.apply_precond(r, 500, only_block=blk)
    assert rel(got, c2abi(want, r.shape)) < 1e-9
    # numpy oracle: same block, PAD and the negative control
    Atr = dense_of(lambda v: a.apply_A_block(v, blk, "TRUNC"), n)
    Apad = dense_of(lambda v: a.apply_A_block(v, blk, "PAD"), n)
    assert np.abs(Apad - As).max() < 1e-12
    assert np.abs(Atr - As).max() > 1e-3        # PAPER.md:127 eq. 11: hop-wise truncation drops snake terms


def test_ps_equals_pad_iff_no_wrap():
    """R10: PS == PAD when L-B >= 4 in every cut direction; they differ on 4^4 with 2^4 blocks (C1 geometry)."""
    dims, Ls, block = (8, 8, 2, 2), 2, (4, 4, 2, 2)
    a, _ = pair(dims, Ls, 0.05, block)
    v = synth.gaussian_spinor_abi(dims, Ls, 3)
    for blk in (0, 3):
        assert rel(a.apply_A_block(v, blk, "PS"), a.apply_A_block(v, blk, "PAD")) < 1e-13
    dims, block = (4, 4, 4, 4), (2, 2, 2, 2)
    a, _ = pair(dims, Ls, 0.05, block)
    v = synth.gaussian_spinor_abi(dims, Ls, 3)
    assert rel(a.apply_A_block(v, 5, "PS"), a.apply_A_block(v, 5, "PAD")) > 1e-4


def test_uncut_block_is_global_operator():
    dims, Ls = (4, 2, 2, 4), 2
    a, c = pair(dims, Ls, 0.05, dims)
    v = synth.gaussian_spinor_abi(dims, Ls, 3)
    assert rel(c.apply_A_block(v, 0), c.apply_MdagM(v)) < 1e-14
    assert rel(a.apply_A_block(v, 0), a.apply_MdagM(v)) < 1e-14


def test_precond_scale_equivariance_zero_input_and_block_independence():
    dims, Ls, block = (4, 4, 4, 4), 2, (2, 2, 4, 4)
    a, c = pair(dims, Ls, 0.05, block)
    r = synth.gaussian_spinor_abi(dims, Ls, 3)
    z = c.apply_precond(r, 3)
    assert rel(c.apply_precond(1e-7 * r, 3), 1e-7 * z) < 1e-12        # R13: z(lambda r) = lambda z(r)
    assert np.all(c.apply_precond(np.zeros_like(r), 3) == 0)           # zero in -> zero out, no NaN
    assert np.all(a.apply_precond(np.zeros_like(r), 3) == 0)
    # per-block scalars: scaling ONE block's input scales only that block's output
    zs = [c.apply_precond(r, 3, only_block=i) for i in range(c.num_blocks)]
    assert rel(sum(zs), z) < 1e-14
    r2 = r.copy().reshape(Ls, -1, 24)
    sup0 = np.abs(zs[0].reshape(Ls, -1, 24)).sum(axis=(0, 2)) > 0
    r2[:, sup0] *= 1e3
    z2 = c.apply_precond(r2.reshape(r.shape), 3)
    assert rel(z2, z + (1e3 - 1) * zs[0]) < 1e-12


def test_mspcg_fewer_outer_iterations_and_snake_terms_help():
    """PAPER.md:190 (fewer outer iterations) and PAPER.md:129 (snake terms crucial) -- qualitative, tiny lattice."""
    dims, Ls, block = (8, 4, 2, 2), 4, (4, 4, 2, 2)
    a, c = pair(dims, Ls, 0.01, block, eps=0.25)
    b = synth.gaussian_spinor_abi(dims, Ls, 2)
    x0, s0 = c.solve(b, tol=1e-9)
    x1, s1 = c.solve(b, tol=1e-9, use_precond=True, n_inner=6)
    assert s1["converged"] and s0["converged"]
    assert s1["iters"] < 0.6 * s0["iters"]
    assert rel(x1, x0) < 1e-7
    assert s1["inner_applies"] == 6 * c.num_blocks * s1["iters"]   # z0 + one per iteration but the last
    # numpy oracle with the hop-wise truncated blocks (negative control) needs more outer iterations
    h = []
    xt, st = a.solve(b, tol=1e-9, use_precond=True, n_inner=6, variant="TRUNC", max_iter=s0["iters"])
    assert st["iters"] > s1["iters"]


def test_sloppy_outer_with_reliable_updates_reaches_fp64_residual():
    """PAPER.md:283 + R17: fp32-rounded iteration with fp64 residual replacement converges to 1e-10."""
    dims, Ls, block = (4, 4, 2, 2), 2, (2, 2, 2, 2)
    a, _ = pair(dims, Ls, 0.02, block)
    b = synth.gaussian_spinor_abi(dims, Ls, 2)
    x_ref, s_ref = a.solve(b, tol=1e-10)
    x, st = a.solve(b, tol=1e-10, sloppy=np.complex64, delta=0.1)
    assert st["converged"] and st["true_res"] <= 1e-10
    assert st["reliable_updates"] >= 3
    assert rel(x, x_ref) < 1e-8
    x, st = a.solve(b, tol=1e-10, sloppy=np.complex64, use_precond=True, n_inner=3)
    assert st["converged"] and st["true_res"] <= 1e-10 and rel(x, x_ref) < 1e-8
    # b = 0 -> x = 0 in 0 iterations (R15); x0 = solution -> 0 iterations
    x, st = a.solve(np.zeros_like(b))
    assert st["iters"] == 0 and np.all(x == 0)
    x, st = a.solve(b, tol=1e-9, x0_abi=x_ref)
    assert st["iters"] == 0 and st["converged"]
