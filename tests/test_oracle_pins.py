"""Pins for the CPU oracle (oracle/): what the paper and the mathematics fix, none of it from the CUDA path.

Each test names the passage (PAPER.md line) or DESIGN.md reading it pins.  CPU only.
"""
import itertools
import os

import numpy as np
import pytest

from oracle import Oracle, mdwf, solvers
from oracle.cbind import OracleC
from paper_2104_05615_b200 import synth

MOB = dict(b=1.5, c=0.5, M5=1.8)
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rel(a, b):
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b))


def make(dims, Ls, mf, block=None, eps=0.3, seed=5, unit=False, tb=-1, cls=Oracle):
    U = synth.unit_links(dims) if unit else synth.random_su3_links(dims, eps, seed)
    o = cls(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf, block)
    o.load_gauge(synth.gauge_natural_to_abi(U, dims), tb)
    return o, U


# ---------------------------------------------------------------- R2 gamma algebra
@pytest.mark.parametrize("which", ["numpy", "c"])
def test_gamma_algebra(which):
    g = mdwf.GAMMA if which == "numpy" else OracleC((2, 2, 2, 2), 2, 1.5, 0.5, 1.8, 0.1).gamma()
    for m in range(4):
        assert np.allclose(g[m], g[m].conj().T)
        for n in range(4):
            assert np.allclose(g[m] @ g[n] + g[n] @ g[m], 2.0 * (m == n) * np.eye(4))
    g5 = g[0] @ g[1] @ g[2] @ g[3]
    assert np.allclose(g5, np.diag([1, 1, -1, -1]))
    for m in range(4):
        assert np.allclose(g5 @ g[m] + g[m] @ g5, 0)


# ---------------------------------------------------------------- R4 M5^-1 closed form
@pytest.mark.parametrize("Ls,mf", [(8, 0.01), (16, 0.002), (12, 0.005), (4, 0.3), (6, 1.0)])
def test_m5inv_closed_form_vs_linalg(Ls, mf):
    mob = mdwf.Mobius(Ls, mf=mf, **MOB)
    A = mob.m5_plus()
    assert np.allclose(mob.m5inv_plus_closed_form(), np.linalg.inv(A), rtol=1e-13, atol=1e-16)
    assert np.allclose(mob.m5inv_plus_closed_form() @ A, np.eye(Ls), atol=1e-15)
    oc = OracleC((2, 2, 2, 2), Ls, MOB["b"], MOB["c"], MOB["M5"], mf)
    assert np.allclose(oc.matrix("m5inv"), np.linalg.inv(oc.matrix("m5")), rtol=1e-13, atol=1e-16)
    assert np.allclose(oc.matrix("m5"), A)
    assert np.allclose(oc.matrix("mphi"), mob.mphi_plus())


def test_m5inv_golden_first_column():
    gold = np.loadtxt(os.path.join(GOLD, "m5inv_first_column.txt"))
    mob = mdwf.Mobius(16, mf=0.002, **MOB)
    assert np.allclose(mob.m5inv_plus_closed_form()[:5, 0], gold, rtol=1e-2)
    oc = OracleC((2, 2, 2, 2), 16, MOB["b"], MOB["c"], MOB["M5"], 0.002)
    assert np.allclose(oc.matrix("m5inv")[:5, 0], gold, rtol=1e-2)


def test_m5_structure_matches_L_definition():
    """R1/R3: alpha + beta*L built from the slice-by-slice definition of L equals the chirality-block form."""
    rng = np.random.default_rng(0)
    mob = mdwf.Mobius(6, mf=0.37, **MOB)
    psi = rng.standard_normal((6, 2, 2, 2, 2, 4, 3)) + 1j * rng.standard_normal((6, 2, 2, 2, 2, 4, 3))
    assert rel(mdwf.M5(mob, psi), mob.alpha * psi + mob.beta * mdwf.L_op(mob, psi)) < 1e-15
    assert rel(mdwf.Mphi(mob, psi), -0.5 * (mob.b * psi + mob.c * mdwf.L_op(mob, psi))) < 1e-15
    assert rel(mdwf.M5inv(mob, mdwf.M5(mob, psi)), psi) < 1e-14
    assert rel(mdwf.M5inv(mob, mdwf.M5(mob, psi, dagger=True), dagger=True), psi) < 1e-14
    # dagger really is the adjoint
    phi = rng.standard_normal(psi.shape) + 1j * rng.standard_normal(psi.shape)
    for f in (mdwf.M5, mdwf.Mphi, mdwf.M5inv):
        assert abs(np.vdot(phi, f(mob, psi)) - np.vdot(f(mob, phi, dagger=True), psi)) < 1e-11


# ---------------------------------------------------------------- eq. 8 by brute force
def _dense_hop_from_eq8(U, dims):
    """Dense matrix of D^w built literally from PAPER.md:105 eq. 8 with its Kronecker deltas (pure Python loops)."""
    Lx, Ly, Lz, Lt = dims
    V = Lx * Ly * Lz * Lt
    ext = (Lx, Ly, Lz, Lt)

    def lex(c):
        return c[0] + Lx * (c[1] + Ly * (c[2] + Lz * c[3]))

    D = np.zeros((V, 4, 3, V, 4, 3), dtype=np.complex128)
    for c in itertools.product(range(Lx), range(Ly), range(Lz), range(Lt)):
        x = lex(c)
        for mu in range(4):
            cm = list(c); cm[mu] = (c[mu] - 1) % ext[mu]
            cp = list(c); cp[mu] = (c[mu] + 1) % ext[mu]
            Uxm = U[mu, cm[3], cm[2], cm[1], cm[0]]          # U_{x-mu,mu}
            Ux = U[mu, c[3], c[2], c[1], c[0]]               # U_{x,mu}
            # (1 + gamma_mu) U^dag_{x-mu,mu} delta_{x-mu,y}
            D[x, :, :, lex(cm), :, :] += np.einsum("ij,ab->iajb", np.eye(4) + mdwf.GAMMA[mu], Uxm.conj().T)
            # (1 - gamma_mu) U_{x,mu} delta_{x+mu,y}
            D[x, :, :, lex(cp), :, :] += np.einsum("ij,ab->iajb", np.eye(4) - mdwf.GAMMA[mu], Ux)
    return D.reshape(V * 12, V * 12)


@pytest.mark.parametrize("cls", [Oracle, OracleC])
def test_hop_bruteforce_and_dagger(cls):
    dims, Ls = (2, 4, 2, 4), 2
    U = synth.random_su3_links(dims, 0.7, 3)
    Dm = _dense_hop_from_eq8(U, dims)
    rng = np.random.default_rng(1)
    V = int(np.prod(dims))
    psi = rng.standard_normal((Ls, V, 4, 3)) + 1j * rng.standard_normal((Ls, V, 4, 3))
    want = (Dm @ psi.reshape(Ls, -1).T).T.reshape(Ls, V, 4, 3)
    want_dag = (Dm.conj().T @ psi.reshape(Ls, -1).T).T.reshape(Ls, V, 4, 3)
    full = psi.reshape(Ls, dims[3], dims[2], dims[1], dims[0], 4, 3)
    if cls is Oracle:
        got = mdwf.hop(U, full).reshape(Ls, V, 4, 3)
        got_dag = mdwf.hop(U, full, dagger=True).reshape(Ls, V, 4, 3)
        assert rel(got, want) < 1e-14 and rel(got_dag, want_dag) < 1e-14
    else:
        # Oracle-B exposes only even-parity operators: check D = 1 - M5inv Dw Mphi M5inv Dw Mphi built from the dense hop
        mob = mdwf.Mobius(Ls, mf=0.2, **MOB)
        oc = cls(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.2)
        oc.load_gauge(synth.gauge_natural_to_abi(U, dims), 1)
        v_abi = synth.gaussian_spinor_abi(dims, Ls, 9)
        v = mdwf.unpack_spinor_abi(v_abi, dims, Ls)

        def dense_hop(f, dag):
            M = Dm.conj().T if dag else Dm
            return (M @ f.reshape(Ls, -1).T).T.reshape(f.shape)

        t = dense_hop(mdwf.Mphi(mob, v), False)
        t = dense_hop(mdwf.Mphi(mob, mdwf.M5inv(mob, t)), False)
        Dv = v - mdwf.M5inv(mob, t)
        assert rel(oc.apply_D(v_abi), mdwf.pack_spinor_abi(Dv, dims)) < 1e-14
        t = dense_hop(mdwf.M5inv(mob, v, True), True)
        t = dense_hop(mdwf.M5inv(mob, mdwf.Mphi(mob, t, True), True), True)
        Ddv = v - mdwf.Mphi(mob, t, True)
        assert rel(oc.apply_D(v_abi, dagger=True), mdwf.pack_spinor_abi(Ddv, dims)) < 1e-14


# ---------------------------------------------------------------- R9 free field in momentum space
def test_free_field_momentum_space():
    dims, Ls, mf = (4, 4, 4, 4), 4, 0.05
    mob = mdwf.Mobius(Ls, mf=mf, **MOB)
    U = mdwf.fold_t_boundary(synth.unit_links(dims), -1)
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    rng = np.random.default_rng(2)
    Lmat = np.zeros((Ls, 4, Ls, 4))
    for s in range(Ls):
        # (L psi)_s = P- psi_{s+1} + P+ psi_{s-1} with -mf wraps
        sp, wp = (s + 1, 1.0) if s + 1 < Ls else (0, -mf)
        sm, wm = (s - 1, 1.0) if s >= 1 else (Ls - 1, -mf)
        Lmat[s, :, sp, :] += wp * mdwf.P_MINUS.real
        Lmat[s, :, sm, :] += wm * mdwf.P_PLUS.real
    Lmat = Lmat.reshape(4 * Ls, 4 * Ls)
    worst = 0.0
    for n in itertools.product(range(Lx), range(Ly), range(Lz), range(Lt)):
        p = np.array([2 * np.pi * n[0] / Lx, 2 * np.pi * n[1] / Ly, 2 * np.pi * n[2] / Lz,
                      2 * np.pi * (n[3] + 0.5) / Lt])
        DW = (4 - MOB["M5"] - np.cos(p).sum()) * np.eye(4) + 1j * sum(np.sin(p[m]) * mdwf.GAMMA[m] for m in range(4))
        small = np.kron(np.eye(Ls), MOB["b"] * DW + np.eye(4)) + np.kron(np.eye(Ls), MOB["c"] * DW - np.eye(4)) @ Lmat
        wave = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
        chi = rng.standard_normal((Ls, 4, 3)) + 1j * rng.standard_normal((Ls, 4, 3))
        psi = wave[None, ..., None, None] * chi[:, None, None, None, None, :, :]
        got = mdwf.D_dw(mob, U, psi)
        want_chi = (small @ chi.reshape(4 * Ls, 3)).reshape(Ls, 4, 3)
        want = wave[None, ..., None, None] * want_chi[:, None, None, None, None, :, :]
        worst = max(worst, rel(got, want))
    assert worst < 1e-13
    # eigenvalues of D_W(p): W(p) +- i sqrt(sum sin^2)
    ev = np.linalg.eigvals(DW)
    W = 4 - MOB["M5"] - np.cos(p).sum()
    assert np.allclose(sorted(ev.imag), sorted([-np.sqrt((np.sin(p) ** 2).sum())] * 2 + [np.sqrt((np.sin(p) ** 2).sum())] * 2))
    assert np.allclose(ev.real, W)


def test_textbook_form_and_shamir_limit():
    dims, Ls = (4, 2, 2, 4), 4
    U = mdwf.fold_t_boundary(synth.random_su3_links(dims, 0.5, 4), -1)
    rng = np.random.default_rng(3)
    psi = rng.standard_normal((Ls, 4, 2, 2, 4, 4, 3)) + 1j * rng.standard_normal((Ls, 4, 2, 2, 4, 4, 3))
    mob = mdwf.Mobius(Ls, mf=0.1, **MOB)
    assert rel(mdwf.D_dw(mob, U, psi), mdwf.D_dw_textbook(mob, U, psi)) < 1e-14
    sh = mdwf.Mobius(Ls, b=1.0, c=0.0, M5=1.8, mf=0.1)
    want = (4 - 1.8) * psi - 0.5 * mdwf.hop(U, psi) + psi - mdwf.L_op(sh, psi)   # D_W + 1 - L
    assert rel(mdwf.D_dw(sh, U, psi), want) < 1e-14


def test_gamma5_hermiticity_and_schur():
    dims, Ls = (4, 2, 4, 2), 4
    o, U = make(dims, Ls, 0.07)
    mob, Uf = o.mob, o.U
    rng = np.random.default_rng(6)
    shp = (Ls, 2, 4, 2, 4, 4, 3)
    u = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
    v = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)

    def G5R(f):  # gamma5 times the reflection s -> Ls-1-s
        g = f[::-1].copy()
        g[..., 2:4, :] *= -1
        return g

    # gamma5-R hermiticity D^dag = G D G holds for the Shamir kernel (c = 0).  For c != 0, L and D_W do not
    # commute, so only D_-^-1 D_DW is G-hermitian (DESIGN.md corrects SURVEY.md on this); what must hold for
    # any b, c is  G D_DW(b,c) G = [(b D_W + 1) + L (c D_W - 1)]^dag, checked below through inner products.
    sh = mdwf.Mobius(Ls, b=1.0, c=0.0, M5=1.8, mf=0.07)
    lhs = np.vdot(u, mdwf.D_dw(sh, Uf, v))             # <u, D v>
    rhs = np.vdot(G5R(mdwf.D_dw(sh, Uf, G5R(u))), v)   # <G D G u, v>  => D^dag = G D G
    assert abs(lhs - rhs) / abs(lhs) < 1e-13
    DW = lambda f: (4 - mob.M5) * f - 0.5 * mdwf.hop(Uf, f)
    other = lambda f: mob.b * DW(f) + f + mdwf.L_op(mob, mob.c * DW(f) - f)   # (b D_W + 1) + L (c D_W - 1)
    lhs = np.vdot(G5R(mdwf.D_dw(mob, Uf, G5R(u))), v)
    rhs = np.vdot(u, other(v))
    assert abs(lhs - rhs) / abs(lhs) < 1e-13
    # Schur identity (R5): psi_o = -M5inv M4oe psi_e  =>  full operator gives (M5 D psi_e, 0)
    ve = mdwf.unpack_spinor_abi(synth.gaussian_spinor_abi(dims, Ls, 1), dims, Ls)
    vo = -mdwf.M5inv(mob, mdwf.hop(Uf, mdwf.Mphi(mob, ve)))
    full = mdwf.D_dw(mob, Uf, ve + vo)
    odd = synth.parity_mask(dims)
    assert np.linalg.norm(full[:, odd]) / np.linalg.norm(full) < 1e-14
    want = mdwf.M5(mob, mdwf.D_eo(mob, Uf, ve))
    assert rel(full[:, ~odd], want[:, ~odd]) < 1e-14
    # D_eo_dag is the adjoint of D_eo; D^dag D Hermitian positive
    a = mdwf.unpack_spinor_abi(synth.gaussian_spinor_abi(dims, Ls, 2), dims, Ls)
    b = mdwf.unpack_spinor_abi(synth.gaussian_spinor_abi(dims, Ls, 3), dims, Ls)
    assert abs(np.vdot(a, mdwf.D_eo(mob, Uf, b)) - np.vdot(mdwf.D_eo_dag(mob, Uf, a), b)) < 1e-10
    Ab = mdwf.MdagM(mob, Uf, b)
    assert abs(np.vdot(a, Ab) - np.conj(np.vdot(b, mdwf.MdagM(mob, Uf, a)))) < 1e-10
    assert abs(np.vdot(b, Ab).real - np.linalg.norm(mdwf.D_eo(mob, Uf, b)) ** 2) < 1e-9
    assert abs(np.vdot(b, Ab).imag) < 1e-10


def test_structure_commutators():
    """links act only on colour; D^w diagonal in s; 5D operators diagonal in 4D and colour."""
    dims, Ls = (2, 4, 2, 4), 4
    U = synth.random_su3_links(dims, 0.4, 8)
    mob = mdwf.Mobius(Ls, mf=0.1, **MOB)
    rng = np.random.default_rng(5)
    shp = (Ls, 4, 2, 4, 2, 4, 3)
    psi = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
    assert rel(mdwf.hop(U, np.roll(psi, 1, axis=0)), np.roll(mdwf.hop(U, psi), 1, axis=0)) < 1e-15
    g = synth.random_su3_field((2, 2, 2, 2), 1)[0, 0, 0, 0]
    rot = lambda f: np.einsum("ab,...b->...a", g, f)
    for f in (mdwf.M5, mdwf.Mphi, mdwf.M5inv):
        assert rel(f(mob, rot(psi)), rot(f(mob, psi))) < 1e-14
    # D^w Mphi != Mphi D^w (gamma_mu and gamma5 anticommute): the order of eq. 7 matters
    assert rel(mdwf.hop(U, mdwf.Mphi(mob, psi)), mdwf.Mphi(mob, mdwf.hop(U, psi))) > 1e-2


@pytest.mark.parametrize("cls", [Oracle, OracleC])
def test_gauge_covariance(cls):
    dims, Ls, block = (4, 4, 4, 4), 2, (2, 2, 4, 4)
    U = synth.random_su3_links(dims, 0.4, 11)
    g = synth.random_su3_field(dims, 12)
    U2 = synth.gauge_transform_links(U, g)
    v = synth.gaussian_spinor_abi(dims, Ls, 4)
    v2 = synth.gauge_transform_spinor_abi(v, g, dims)
    o1 = cls(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.05, block)
    o2 = cls(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.05, block)
    o1.load_gauge(synth.gauge_natural_to_abi(U, dims), -1)
    o2.load_gauge(synth.gauge_natural_to_abi(U2, dims), -1)
    assert rel(o2.apply_MdagM(v2), synth.gauge_transform_spinor_abi(o1.apply_MdagM(v), g, dims)) < 1e-13
    z1 = o1.apply_precond(v, 3)
    z2 = o2.apply_precond(v2, 3)
    assert rel(z2, synth.gauge_transform_spinor_abi(z1, g, dims)) < 1e-11
    # and the transformed field really is different
    assert rel(o2.apply_MdagM(v), o1.apply_MdagM(v)) > 1e-2


def test_antiperiodic_time_matters_and_sign_fold():
    dims, Ls = (2, 2, 2, 4), 2
    U = synth.random_su3_links(dims, 0.3, 1)
    Ua = synth.gauge_natural_to_abi(U, dims)
    v = synth.gaussian_spinor_abi(dims, Ls, 1)
    outs = {}
    for tb in (+1, -1):
        o = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.1)
        o.load_gauge(Ua, tb)
        outs[tb] = o.apply_MdagM(v)
    assert rel(outs[1], outs[-1]) > 1e-3
    U2 = U.copy(); U2[3, -1] *= -1
    o = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.1)
    o.load_gauge(synth.gauge_natural_to_abi(U2, dims), +1)
    assert rel(o.apply_MdagM(v), outs[-1]) < 1e-15
