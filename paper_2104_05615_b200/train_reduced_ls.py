"""Set-up tool: train the reduced-Ls transfer matrix T of PAPER.md:299-326 (eq. 20-22) with the library's own kernels.

    from paper_2104_05615_b200.train_reduced_ls import train
    T_abi, info = train(dims, Ls, mob, mf, block, U_abi, b_abi, Ls_hat, mu, n_inner)

Recipe: the training vectors v_i are residual vectors r_k of a full-Ls MSPCG solve of the same system
(here: r_k = b - A x_k with x_k the iterate after k outer iterations, k spread over the first `span` iterations); T starts
from the untrained selection matrix (reading R20) and is updated by line search with momentum on chi2 (eq. 22).  Training
runs in a context with fp32 inner storage (the loss of eq. 22 is not evaluated in fp16); the result is used in any context.
Argument marshalling only: every operator application, inner product and outer product runs in libmspcg's kernels.
"""
from __future__ import annotations

import numpy as np

from .binding import F32, F64, Mspcg


def initial_T_abi(Ls, Lh):
    """Spin identity, keeps the Lh/2 slices next to each domain wall (reading R20).  float64 [4*Lh][4*Ls][re,im]."""
    T = np.zeros((Lh, 4, Ls, 4, 2))
    for a in range(Lh):
        s = a if a < Lh // 2 else Ls - Lh + a
        for m in range(4):
            T[a, m, s, m, 0] = 1.0
    return T.reshape(-1)


def residual_vectors(g, d_b, n_inner, n_vec, span):
    """r_k = b - A x_k of a full-Ls MSPCG run (fp64 operator), k = span/n_vec, 2 span/n_vec, ...; normalised.  torch only concatenates."""
    import torch
    out = []
    for j in range(1, n_vec + 1):
        k = max(1, (span * j) // n_vec)
        x, _ = g.solve(d_b, tol=1e-14, max_iter=k, use_precond=True, n_inner=n_inner, sloppy_prec=F32)
        out.append(g.residual(d_b, x, normalise=True)[0])   # formed and normalised inside the library (mspcg_residual)
    return torch.cat(out)


def train(dims, Ls, mob, mf, block, U_abi, b_abi, Ls_hat, mu, n_inner, n_vec=8, span=120, n_steps=20, momentum=0.5, T0_abi=None):
    import torch
    g = Mspcg(dims, Ls, mob["b"], mob["c"], mob["M5"], mf, block)
    g.set_reduced_ls(Ls_hat, initial_T_abi(Ls, Ls_hat) if T0_abi is None else T0_abi, mu)
    g.configure(F32, F32, 18)
    g.load_gauge(U_abi, -1)
    d_b = torch.as_tensor(np.ascontiguousarray(b_abi, dtype=np.float64).reshape(-1)).cuda()
    vs = residual_vectors(g, d_b, n_inner, n_vec, span)
    T, hist = g.train_T(vs, n_inner, n_steps, momentum)
    g.close()
    return T, dict(chi2=hist, n_vec=n_vec, n_steps=n_steps, mu=mu)
