"""Pins for the oracle's full 4-step solve: source preparation (eq. 6), the CGNR right-hand
side (eq. 9) and the odd-site reconstruction (second row of PAPER.md:91 eq. 4).

What pins them is a dense direct solve of the unpreconditioned 2x2 system of eq. (4) on a tiny lattice: the operator D_dw
is pinned on its own (free-field momentum space, textbook form; tests/test_oracle_pins.py), its dense inverse knows nothing
of the Schur complement, and a dropped factor, a wrong sign or a swapped parity in eq. (5)/(6) fails one of the checks.  CPU only.
"""
import numpy as np

from oracle import Oracle, mdwf, solvers
from paper_2104_05615_b200 import synth

MOB = dict(b=1.5, c=0.5, M5=1.8)


def rel(a, b):
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b))


def test_prepared_source_and_reconstruction_vs_dense_direct_solve():
    dims, Ls, mf = (2, 2, 2, 2), 4, 0.05
    o = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf)
    o.load_gauge(synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.3, 3), dims), -1)
    mob, U = o.mob, o.U
    shp = (Ls, 2, 2, 2, 2, 4, 3)
    n = int(np.prod(shp))
    Dm = np.empty((n, n), dtype=np.complex128)
    for j in range(n):
        e = np.zeros(n, dtype=np.complex128); e[j] = 1.0
        Dm[:, j] = mdwf.D_dw(mob, U, e.reshape(shp)).reshape(-1)
    rng = np.random.default_rng(8)
    phi = rng.standard_normal(shp) + 1j * rng.standard_normal(shp)
    psi = np.linalg.solve(Dm, phi.reshape(-1)).reshape(shp)              # the solution of eq. (4), no even-odd anywhere
    odd = synth.parity_mask(dims)
    split = lambda f: (np.where(odd[None, ..., None, None], 0, f), np.where(odd[None, ..., None, None], f, 0))
    phi_e, phi_o = split(phi)
    psi_e, psi_o = split(psi)
    # eq. (5)/(6): the even part of the solution solves D psi_e = phihat_e
    hat = mdwf.prepare_source(mob, U, phi_e, phi_o)
    assert np.linalg.norm(hat[:, odd]) == 0.0
    assert rel(mdwf.D_eo(mob, U, psi_e), hat) < 1e-11
    # second row of eq. (4): the odd part follows from the even part
    assert rel(mdwf.reconstruct_odd(mob, U, psi_e, phi_o), psi_o) < 1e-11
    # eq. (9): CG on the normal equations with the prepared right-hand side reaches the same even part
    rhs = mdwf.normal_rhs(mob, U, phi_e, phi_o)
    x, st = solvers.pcg(lambda v: mdwf.MdagM(mob, U, v), rhs, None, 1e-13, 5000)
    assert st["converged"]
    assert rel(x, psi_e) < 1e-9
    full = mdwf.D_dw(mob, U, x + mdwf.reconstruct_odd(mob, U, x, phi_o))
    assert rel(full, phi) < 1e-9
    # negative controls: the plausible mistakes do not pass
    wrong_sign = mdwf.M5inv(mob, phi_e) + mdwf.M5inv(mob, mdwf.M4(mob, U, mdwf.M5inv(mob, phi_o)))
    assert rel(mdwf.D_eo(mob, U, psi_e), wrong_sign) > 1e-2
    no_inner_m5inv = mdwf.M5inv(mob, phi_e) - mdwf.M5inv(mob, mdwf.M4(mob, U, phi_o))
    assert rel(mdwf.D_eo(mob, U, psi_e), no_inner_m5inv) > 1e-2


def test_abi_facade_round_trip():
    """Oracle.prepare_source / reconstruct_odd / apply_full on ABI arrays: solve, reconstruct, apply eq. (4), get the source back."""
    dims, Ls, mf = (4, 2, 2, 4), 4, 0.1
    o = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf)
    o.load_gauge(synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.3, 4), dims), -1)
    phi_e = synth.gaussian_spinor_abi(dims, Ls, 31)
    phi_o = synth.gaussian_spinor_abi(dims, Ls, 32)
    # even/odd ABI vectors unpack onto complementary supports
    fe, fo = o.unpack(phi_e), o.unpack_odd(phi_o)
    odd = synth.parity_mask(dims)
    assert np.linalg.norm(fe[:, odd]) == 0.0 and np.linalg.norm(fo[:, ~odd]) == 0.0
    assert np.array_equal(o.pack_odd(fo), phi_o)
    hat, rhs = o.prepare_source(phi_e, phi_o)
    assert rel(o.apply_D(hat, dagger=True), rhs) < 1e-14
    x, st = o.solve(rhs, tol=1e-12)
    assert st["converged"]
    psi_o = o.reconstruct_odd(x, phi_o)
    out_e, out_o = o.apply_full(x, psi_o)
    assert rel(out_e, phi_e) < 1e-9 and rel(out_o, phi_o) < 1e-9
