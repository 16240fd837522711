"""Training of the reduced-Ls transfer matrix (eq. 22) -- the library against oracle/reduced_ls.py on the same
seeded inputs: loss, gradient (every entry) and the T sequence of the line search with momentum.

What this pins and what it does not.  The loss chi2 (eq. 22) and its analytic gradient are definitions: the oracle's gradient is pinned by
central finite differences (tests/test_oracle_reduced_ls.py), so the first two tests are parity proper.  The STEP RULE (five samples at
eta0 (0, 1/2, 1, 3/2, 2), quartic fit, momentum dropped and eta0 quartered after a step without decrease) is a reading of the paper's two words
"line search" and "momentum" (parity unpinned) that the oracle and the library implement alike -- the T-sequence
test shows that the two follow the same rule to rounding, not that the rule is the paper's."""
import numpy as np
import pytest

from paper_2104_05615_b200 import F64, Mspcg, synth

pytestmark = pytest.mark.gpu
MOB = dict(b=1.5, c=0.5, M5=1.8)


def rel(a, b):
    a, b = np.asarray(a, dtype=np.float64).reshape(-1), np.asarray(b, dtype=np.float64).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _setup(dims, Ls, Lh, block, mu, seed=31):
    import torch
    from oracle import Oracle, reduced_ls
    U = synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.3, 5), dims)
    full = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.05, block)
    full.load_gauge(U, -1)
    hat = Oracle(dims, Lh, MOB["b"], MOB["c"], MOB["M5"], 0.05, block)
    hat.load_gauge(U, -1)
    rng = np.random.default_rng(seed)
    T = reduced_ls.initial_T(Ls, Lh) + 0.05 * (rng.standard_normal((Lh, 4, Ls, 4)) + 1j * rng.standard_normal((Lh, 4, Ls, 4)))
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.05, block)
    g.set_reduced_ls(Lh, reduced_ls.T_to_abi(T), mu)
    g.configure(F64, F64, 18)
    g.load_gauge(U, -1)
    Pf, Ph = full.precond_obj(), hat.precond_obj()

    def M_apply(w):
        out = np.zeros_like(w)
        for o in Pf.origins:
            out += Pf.apply_A_block(o, w)
        return out
    vs_abi = [synth.gaussian_spinor_abi(dims, Ls, 40 + i) for i in range(2)]
    vs = [full.unpack(v) for v in vs_abi]
    dv = torch.as_tensor(np.concatenate([v.reshape(-1) for v in vs_abi])).cuda()
    return reduced_ls, M_apply, Ph, T, vs, dv, g


def test_loss_and_gradient_match_the_oracle():
    dims, Ls, Lh, block, mu, k = (4, 4, 2, 4), 8, 4, (2, 2, 2, 2), 0.3, 3
    rl, M_apply, Ph, T, vs, dv, g = _setup(dims, Ls, Lh, block, mu)
    val_o, G_o = rl.chi2_and_gradient(M_apply, lambda r: Ph(r, k), T, mu, vs)
    val, G = g.train_eval(dv, k)
    assert abs(val - val_o) <= 1e-9 * val_o
    assert rel(G, rl.T_to_abi(G_o)) <= 1e-8
    val2, _ = g.train_eval(dv, k, want_grad=False)
    assert abs(val2 - val) <= 1e-12 * val      # atomics: summation order differs between runs


def test_training_steps_follow_the_oracle_and_reduce_the_loss():
    dims, Ls, Lh, block, mu, k = (4, 2, 2, 4), 6, 4, (2, 2, 2, 2), 0.4, 4
    rl, M_apply, Ph, T, vs, dv, g = _setup(dims, Ls, Lh, block, mu)
    Ahat = lambda r: Ph(r, k)
    To, hist_o = rl.train(M_apply, Ahat, T, mu, vs, 2, 0.5)
    Tg, hist = g.train_T(dv, k, 2, momentum=0.5)
    assert np.all(np.diff(hist) < 0)
    assert rel(hist, hist_o) <= 1e-6
    assert rel(Tg, rl.T_to_abi(To)) <= 1e-5
    # the context now applies the trained T
    val, _ = g.train_eval(dv, k, want_grad=False)
    assert abs(val - hist[-1]) <= 1e-12 * val
