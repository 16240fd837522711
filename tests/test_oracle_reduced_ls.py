"""Pins of oracle/reduced_ls.py (eq. 19-21) against special cases written with explicit indexing."""
import numpy as np

from oracle import Oracle, mdwf, reduced_ls, solvers
from paper_2104_05615_b200 import synth

DIMS, BLOCK, LS = (4, 4, 4, 4), (2, 2, 4, 4), 4
MOB = dict(b=1.5, c=0.5, M5=1.8, mf=0.05)


def _setup(Ls_hat, DIMS=DIMS, BLOCK=BLOCK):
    U = synth.gauge_natural_to_abi(synth.random_su3_links(DIMS, 0.3, 3), DIMS)
    full = Oracle(DIMS, LS, MOB["b"], MOB["c"], MOB["M5"], MOB["mf"], BLOCK)
    full.load_gauge(U, -1)
    hat = Oracle(DIMS, Ls_hat, MOB["b"], MOB["c"], MOB["M5"], MOB["mf"], BLOCK)
    hat.load_gauge(U, -1)
    r = full.unpack(synth.gaussian_spinor_abi(DIMS, LS, 4))
    return full, hat, r


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def test_identity_T_reproduces_the_full_preconditioner():
    """with Ls_hat = Ls, Mhat = M and T = 1; then eq. 20 at mu = 0 is eq. 19."""
    full, hat, r = _setup(LS)
    T = reduced_ls.initial_T(LS, LS)
    assert np.array_equal(T.reshape(4 * LS, 4 * LS), np.eye(4 * LS))
    z = reduced_ls.ReducedLsPrecond(hat.precond_obj(), T, 0.0)(r, 3)
    assert rel(z, full.precond_obj()(r, 3)) <= 1e-14
    z2 = reduced_ls.ReducedLsPrecond(hat.precond_obj(), T, 0.37)(r, 3)
    assert rel(z2 - z, 0.37 * r) <= 1e-13


def test_slice_permutation_gamma5_and_phase():
    full, hat, r = _setup(LS)
    P = hat.precond_obj()
    ref = lambda v: P(v, 2)
    # cyclic slice shift (not an involution): (T v)_a = v_{(a+1) mod Ls}; T^dag w puts w_a back at slice a+1
    T = np.zeros((LS, 4, LS, 4), dtype=complex)
    for a in range(LS):
        for m in range(4):
            T[a, m, (a + 1) % LS, m] = 1.0
    z = reduced_ls.ReducedLsPrecond(P, T, 0.0)(r, 2)
    assert rel(z, np.roll(ref(np.roll(r, -1, axis=0)), 1, axis=0)) <= 1e-14
    assert rel(np.roll(ref(np.roll(r, 1, axis=0)), -1, axis=0), z) > 1e-3      # the transposed map differs
    # T = 1 (x) gamma5 = sign flip of spin components 2, 3
    T = np.zeros((LS, 4, LS, 4), dtype=complex)
    for a in range(LS):
        for m in range(4):
            T[a, m, a, m] = 1.0 if m < 2 else -1.0
    g5 = np.array([1, 1, -1, -1.0])[:, None]
    assert rel(reduced_ls.ReducedLsPrecond(P, T, 0.0)(r, 2), g5 * ref(g5 * r)) <= 1e-14
    # a spin-mixing unitary on one slice pair: (T v)_{a, m} = sum_n G[m, n] v_{a, n} with G = gamma_1 (Hermitian)
    G = mdwf.GAMMA[0]
    T = np.einsum("ab,mn->ambn", np.eye(LS), G).astype(complex)
    gv = lambda v: np.einsum("mn,stzyxnc->stzyxmc", G, v)
    assert rel(reduced_ls.ReducedLsPrecond(P, T, 0.0)(r, 2), gv(ref(gv(r)))) <= 1e-14
    # T = i: T^dag Mhat^-1 T = (-i) CG(i r) = CG(r) (the block CG is homogeneous of degree one for complex scalars)
    T = 1j * reduced_ls.initial_T(LS, LS)
    assert rel(reduced_ls.ReducedLsPrecond(P, T, 0.0)(r, 2), ref(r)) <= 1e-13


def test_rectangular_slice_selection():
    """Ls_hat < Ls, T = initial_T: T picks slices (0, Ls-1) for Ls_hat = 2; T^dag scatters them back into zeros."""
    full, hat, r = _setup(2)
    T = reduced_ls.initial_T(LS, 2)
    P = hat.precond_obj()
    z = reduced_ls.ReducedLsPrecond(P, T, 0.25)(r, 3)
    sel = [0, LS - 1]
    zh = P(r[sel], 3)
    want = 0.25 * r
    want[sel] += zh
    assert rel(z, want) <= 1e-14
    # ABI round trip of T
    assert np.array_equal(reduced_ls.T_from_abi(reduced_ls.T_to_abi(T), 2, LS), T)


def test_reduced_pcg_reaches_the_same_solution():
    """eq. 20 only changes the path: PCG with the reduced-Ls preconditioner solves the same SPD system (mu > 0)."""
    full, hat, r = _setup(2, (2, 2, 2, 4), (2, 2, 2, 2))
    A = lambda v: mdwf.MdagM(full.mob, full.U, v)
    pre = reduced_ls.ReducedLsPrecond(hat.precond_obj(), reduced_ls.initial_T(LS, 2), 0.5)
    x0, s0 = solvers.pcg(A, r, None, 1e-9)
    x1, s1 = solvers.pcg(A, r, lambda v: pre(v, 3), 1e-9)
    assert rel(x1, x0) <= 1e-7 and s1["converged"]


# ---- training of T (eq. 22; reading R20) ------------------------------------------------------------
def _train_setup(Ls_hat, k):
    dims, block = (2, 2, 2, 4), (2, 2, 2, 2)
    full, hat, r = _setup(Ls_hat, dims, block)
    Pf, Ph = full.precond_obj(), hat.precond_obj()

    def M_apply(w):   # (+)_s A_s w
        out = np.zeros_like(w)
        for o in Pf.origins:
            out += Pf.apply_A_block(o, w)
        return out
    vs = [r]
    return M_apply, (lambda rh: Ph(rh, k)), vs


def test_chi2_vanishes_for_identity_T():
    """Ls_hat = Ls => Mhat = M, optimal T = 1, optimal chi2 = 0 (mu = 0, converged block solve)."""
    M_apply, Ahat, vs = _train_setup(LS, 160)
    c0 = reduced_ls.chi2(M_apply, Ahat, reduced_ls.initial_T(LS, LS), 0.0, vs)
    norm = sum(np.vdot(v, v).real for v in vs)
    assert c0 <= 1e-16 * norm
    # and it does not vanish away from it
    assert reduced_ls.chi2(M_apply, Ahat, 0.9 * reduced_ls.initial_T(LS, LS), 0.0, vs) > 1e-3 * norm


def test_gradient_against_finite_differences_and_line_search():
    M_apply, Ahat, vs = _train_setup(2, 120)      # converged CG: Ahat is linear and Hermitian, as R20 assumes
    rng = np.random.default_rng(8)
    T = reduced_ls.initial_T(LS, 2) + 0.1 * (rng.standard_normal((2, 4, LS, 4)) + 1j * rng.standard_normal((2, 4, LS, 4)))
    mu = 0.3
    val, G = reduced_ls.chi2_and_gradient(M_apply, Ahat, T, mu, vs)
    assert abs(val - reduced_ls.chi2(M_apply, Ahat, T, mu, vs)) <= 1e-12 * val
    for seed in (1,):
        r2 = np.random.default_rng(seed)
        dT = r2.standard_normal(T.shape) + 1j * r2.standard_normal(T.shape)
        h = 1e-5
        fd = (reduced_ls.chi2(M_apply, Ahat, T + h * dT, mu, vs) - reduced_ls.chi2(M_apply, Ahat, T - h * dT, mu, vs)) / (2 * h)
        an = 2.0 * np.vdot(G, dT).real
        assert abs(fd - an) <= 1e-6 * abs(an)
    # the quartic through five points is exact for a linear Ahat: its minimum beats a brute-force scan along -G
    T1, P, v0, eta = reduced_ls.train_step(M_apply, Ahat, T, mu, vs)
    v1 = reduced_ls.chi2(M_apply, Ahat, T1, mu, vs)
    scan = min(reduced_ls.chi2(M_apply, Ahat, T + x * eta * P, mu, vs) for x in (0.9, 1.1))
    assert v1 < v0 and v1 <= scan * (1 + 1e-9)
