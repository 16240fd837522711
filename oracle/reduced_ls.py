"""ORACLE (test infrastructure only) -- the reduced-Ls preconditioner of PAPER.md:299-326 (eq. 19-22).

Plain numpy complex128, written from the paper; shares no code with the CUDA path.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import it.

  eq. 20:  z = (T^dag Mhat^-1 T + mu) r
  eq. 21:  [T v]_{s,mu} = sum_{t,nu} T[s t, mu nu] v[t, nu],  t = 1..Ls, s = 1..Ls_hat,
                          mu, nu spin indices; T is the identity in colour and in the 4D site.
  "Mhat^-1" is the multi-splitting preconditioner built with Ls_hat and the SAME b, c, M5, mf, solved by the same
  fixed number of block CG iterations (reading R19).

Array convention: T[s_hat, spin', s, spin] complex128 (the C-ABI order T_host[4*Ls_hat][4*Ls][re,im] of
include/mspcg.h reshaped); fields psi[s, t, z, y, x, spin, colour] as in oracle/mdwf.py.

Pins (tests/test_oracle_reduced_ls.py): Ls_hat = Ls, T = 1, mu = 0 reproduces the full-Ls preconditioner;
the mu term is exactly mu*r; T = a cyclic slice permutation, T = 1 (x) gamma5, T = i*1 and T = a slice selection
each against the same map written with explicit array indexing (they fail if T and T^dag are exchanged, if the
conjugate is dropped, or if the spin and slice indices are transposed).  initial_T (reading R20: the paper does not
give the starting point of the training) is a convention, not a result: parity unpinned.

Training of T (eq. 22; reading R20): chi2, its gradient with respect to conj(T) and one
line-search step with momentum.  Pins: chi2 = 0 at Ls_hat = Ls, T = 1, mu = 0 with a converged block solve
(PAPER.md:322); the analytic gradient against central finite differences of chi2 in random directions (with a
converged, hence linear and Hermitian, Mhat^-1); the exact quartic line search against a brute-force scan.
"""
from __future__ import annotations

import numpy as np


def apply_T(T, v):
    """eq. 21: (T v)[a, ..., m, c] = sum_{b, n} T[a, m, b, n] v[b, ..., n, c]."""
    return np.einsum("ambn,btzyxnc->atzyxmc", T, v)


def apply_Tdag(T, vh):
    """(T^dag w)[b, ..., n, c] = sum_{a, m} conj(T[a, m, b, n]) w[a, ..., m, c]."""
    return np.einsum("ambn,atzyxmc->btzyxnc", np.conj(T), vh)


def T_from_abi(T_abi, Ls_hat, Ls):
    a = np.asarray(T_abi, dtype=np.float64).reshape(Ls_hat, 4, Ls, 4, 2)
    return a[..., 0] + 1j * a[..., 1]


def T_to_abi(T):
    return np.ascontiguousarray(np.stack([T.real, T.imag], axis=-1).reshape(-1))


def initial_T(Ls, Ls_hat):
    """Reading R20 (paper silent): spin identity; s_hat < Ls_hat/2 <-> s = s_hat, the rest <-> s = Ls - Ls_hat + s_hat
    (keep the slices next to both domain walls).  Ls_hat = Ls gives the identity."""
    T = np.zeros((Ls_hat, 4, Ls, 4), dtype=np.complex128)
    for a in range(Ls_hat):
        s = a if a < Ls_hat // 2 else Ls - Ls_hat + a
        for m in range(4):
            T[a, m, s, m] = 1.0
    return T


class ReducedLsPrecond:
    """eq. 20.  `pre_hat` is the Ls_hat block preconditioner: pre_hat(r_hat, k) -> z_hat (oracle.solvers.BlockPrecond
    built with a Mobius object of Ls_hat)."""

    def __init__(self, pre_hat, T, mu):
        self.pre_hat, self.T, self.mu = pre_hat, np.asarray(T, dtype=np.complex128), float(mu)

    def __call__(self, r, k):
        return apply_Tdag(self.T, self.pre_hat(apply_T(self.T, r), k)) + self.mu * r


# ---------------------------------------------------------------------------------------------------------------
# eq. 22:  chi2(T) = sum_i | M (T^dag Ahat T + mu) v_i - v_i |^2
#   M    = the full-Ls block operator (+)_s A_s (Hermitian),  M_apply(w) -> M w
#   Ahat = Mhat^-1 = the fixed-count block CG at Ls_hat,      Ahat_apply(r_hat) -> z_hat
# Reading R20: for the derivative Ahat is treated as a fixed Hermitian linear operator.  With
#   w = (T^dag Ahat T + mu) v,  e = M w - v,  g = M e,  a = Ahat T v,  c = Ahat T g:
#   d chi2 = 2 Re sum_i [ <c_i, dT v_i> + <a_i, dT g_i> ]   =>   G = d chi2 / d conj(T) = sum_i (c_i v_i^dag + a_i g_i^dag)
# (outer products summed over 4D sites and colour; G has the shape of T).
# ---------------------------------------------------------------------------------------------------------------
def outer_T(x_hat, y):
    """sum over sites and colour of x_hat[a, ..., m, c] conj(y[b, ..., n, c]) -> [a, m, b, n]."""
    return np.einsum("atzyxmc,btzyxnc->ambn", x_hat, np.conj(y))


def chi2_terms(M_apply, Ahat_apply, T, mu, v):
    a = Ahat_apply(apply_T(T, v))
    w = apply_Tdag(T, a) + mu * v
    e = M_apply(w) - v
    return a, w, e


def chi2(M_apply, Ahat_apply, T, mu, vs):
    return float(sum(np.vdot(e, e).real for e in (chi2_terms(M_apply, Ahat_apply, T, mu, v)[2] for v in vs)))


def chi2_and_gradient(M_apply, Ahat_apply, T, mu, vs):
    val, G = 0.0, np.zeros_like(T)
    for v in vs:
        a, w, e = chi2_terms(M_apply, Ahat_apply, T, mu, v)
        val += float(np.vdot(e, e).real)
        g = M_apply(e)
        c = Ahat_apply(apply_T(T, g))
        G += outer_T(c, v) + outer_T(a, g)
    return val, G


def quartic_minimum(etas, vals):
    """chi2(T + eta P) is a quartic in eta when Ahat is linear: fit it through five evaluations and return the minimiser
    of the fit over the sampled interval [etas[0], etas[-1]] ("line search"): the candidates are the real
    stationary points inside the interval and the sample points themselves.  (The fixed-count CG is only approximately
    linear, so the fit is not trusted outside the interval it was measured on.)"""
    etas = np.asarray(etas, dtype=np.float64)
    coef = np.polyfit(etas / etas[-1], np.asarray(vals, dtype=np.float64), 4)
    roots = np.roots(np.polyder(coef))
    cand = [float(x) for x in etas / etas[-1]]
    cand += [r.real for r in roots if abs(r.imag) <= 1e-9 * max(1.0, abs(r.real)) and 0.0 <= r.real <= 1.0]
    return float(min(cand, key=lambda x: np.polyval(coef, x))) * float(etas[-1])


def train_step(M_apply, Ahat_apply, T, mu, vs, direction_prev=None, momentum=0.0, scale=1.0):
    """One step: P = -G + momentum * P_prev; five evaluations at eta0 * (0, 1/2, 1, 3/2, 2); T <- T + eta* P.
    eta0 = scale * chi2 / |G|^2 (the Newton-like scale of a quadratic).  Returns (T_new, P, chi2_before, eta*)."""
    val, G = chi2_and_gradient(M_apply, Ahat_apply, T, mu, vs)
    P = -G if direction_prev is None else -G + momentum * direction_prev
    eta0 = scale * val / float(np.vdot(G, G).real)
    etas = [0.0, 0.5 * eta0, eta0, 1.5 * eta0, 2.0 * eta0]
    vals = [val] + [chi2(M_apply, Ahat_apply, T + h * P, mu, vs) for h in etas[1:]]
    eta = quartic_minimum(etas, vals)
    best = int(np.argmin(vals))
    if eta not in etas and chi2(M_apply, Ahat_apply, T + eta * P, mu, vs) > vals[best]:
        eta = etas[best]          # the fit promised more than the loss delivers: keep the best measured point
    return T + eta * P, P, val, eta


def train(M_apply, Ahat_apply, T, mu, vs, n_steps, momentum):
    """n_steps of train_step.  When a step finds no decrease (eta* = 0) the momentum is dropped and the step scale is
    quartered; after a successful step the scale doubles back towards 1.  Returns (T, [chi2 before each step, final chi2])."""
    P, scale, hist = None, 1.0, []
    for _ in range(n_steps):
        T, P, val, eta = train_step(M_apply, Ahat_apply, T, mu, vs, P, momentum, scale)
        hist.append(val)
        if eta == 0.0:
            P, scale = None, scale * 0.25
        else:
            scale = min(1.0, scale * 2.0)
    hist.append(chi2(M_apply, Ahat_apply, T, mu, vs))
    return T, hist
