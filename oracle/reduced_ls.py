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
give the starting point of the training) is a convention, not a result: parity unpinned.  The training of T
(eq. 22) is not implemented in the oracle.
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
