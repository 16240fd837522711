"""ORACLE (test infrastructure only) -- CG, the multi-splitting preconditioner and MSPCG.

Plain numpy float64/complex128, step by step in the paper's order and notation; shares no
code with the CUDA path.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import it.

Cites: Algorithm 1, eq. 12-14, fixed inner iteration
count, Polak-Ribiere beta eq. 18, reliable updates (PAPER.md:283,
rule = reading R17).  Pins: dense direct solves, "k >= dim block CG = A_s^-1", CG and MSPCG reach
the same x (tests/test_oracle_solvers.py); the outer loop's path (beta) by CG theory: finite termination,
conjugacy, PR = FR for a fixed linear M, iteration counts of a textbook loop (tests/test_oracle_cg_theory.py).
"""
from __future__ import annotations

import numpy as np

from . import mdwf


def rdot(a, b):
    """Real part of the complex inner product <a,b> = sum conj(a) b (R13)."""
    return float(np.vdot(a, b).real)


# ---------------------------------------------------------------------------
# R13 -- fixed-count CG on one block, zero initial guess.
#   x=0; r=r_s; p=r; rho=<r,r>; repeat k times { q=A p; a=rho/<p,q>; x+=a p; r-=a q;
#   rho'=<r,r>; p=r+(rho'/rho) p; rho=rho' }
# rho == 0 or <p,q> <= 0 stops that block early and returns the current x (never NaN).
# ---------------------------------------------------------------------------
def cg_fixed(apply_A, r_in, k):
    x = np.zeros_like(r_in)
    r = r_in.copy()
    p = r.copy()
    rho = rdot(r, r)
    napply = 0
    for _ in range(k):
        if rho == 0.0:
            break
        q = apply_A(p)
        napply += 1
        pq = rdot(p, q)
        if not pq > 0.0:
            break
        a = rho / pq
        x += a * p
        r -= a * q
        rho_new = rdot(r, r)
        p = r + (rho_new / rho) * p
        rho = rho_new
    return x, napply


class BlockPrecond:
    """M = (+)_s A_s (eq. 14), each block solved by k CG steps from a zero guess (eq. 13)."""

    def __init__(self, mob, U, dims, block, variant="PAD"):
        self.mob, self.U, self.dims, self.block, self.variant = mob, U, tuple(dims), tuple(block), variant
        for L, B in zip(dims, block):
            if L % B or B % 2:
                raise ValueError("block dims must be even and divide the lattice")
        self.origins = mdwf.block_origins(dims, block)
        self.centre = mdwf.box_centre_mask(dims, block)
        self.napply = 0
        self._links = {}

    def _box(self, o):
        if o not in self._links:
            self._links[o] = mdwf.box_links(self.U, self.dims, self.block, o)
        return self._links[o]

    def apply_A_block(self, o, v_full):
        """A_s applied to the block-o part of a full-lattice even field; result on the block, zero elsewhere."""
        out = np.zeros_like(v_full)
        if self.variant == "PAD":
            Ub, per = self._box(o)
            vb = mdwf.box_embed(v_full, self.dims, self.block, o)
            wb = mdwf.A_block_pad(self.mob, Ub, per, vb, self.centre)
            mdwf.box_extract_add(out, wb, self.dims, self.block, o)
            return out
        if self.variant == "PS":
            return mdwf.A_block_ps(self.mob, self.U, self.dims, self.block, o, v_full)
        if self.variant == "TRUNC":
            return mdwf.A_block_hopwise_truncated(self.mob, self.U, self.dims, self.block, o, v_full)
        raise ValueError(self.variant)

    def __call__(self, r_full, k, blocks=None):
        """z = M^-1 r: independent k-step CG per block (own alpha_i, beta_i per block, R13)."""
        z = np.zeros_like(r_full)
        todo = self.origins if blocks is None else [self.origins[i] for i in blocks]
        for o in todo:
            if self.variant == "PAD":
                Ub, per = self._box(o)
                rb = mdwf.box_embed(r_full, self.dims, self.block, o)
                xb, n = cg_fixed(lambda p: mdwf.A_block_pad(self.mob, Ub, per, p, self.centre), rb, k)
                mdwf.box_extract_add(z, xb, self.dims, self.block, o)
            else:
                m = np.zeros_like(r_full)
                mdwf.box_extract_add  # noqa: B018  (kept for symmetry; PS path works on full fields)
                Bx, By, Bz, Bt = self.block
                ox, oy, oz, ot = o
                sl = (slice(None), slice(ot, ot + Bt), slice(oz, oz + Bz), slice(oy, oy + By), slice(ox, ox + Bx))
                m[sl] = r_full[sl]
                xb, n = cg_fixed(lambda p: self.apply_A_block(o, p), m, k)
                z[sl] = xb[sl]
            self.napply += n
        return z


# ---------------------------------------------------------------------------
# Algorithm 1 (r0 = b - A x0 first: R15) with the Polak-Ribiere beta of
# eq. 18 and optional reliable updates (R17).  precond=None gives plain CG (z = r).
# `sloppy` emulates a low-precision iteration by rounding the iterated vectors through that dtype.
# ---------------------------------------------------------------------------
def pcg(apply_A, b, precond=None, tol=1e-10, max_iter=100000, x0=None,
        sloppy=None, delta=0.1, history=None):
    bnorm = np.sqrt(rdot(b, b))
    stats = dict(iters=0, reliable_updates=0, converged=False, breakdown=False)
    if bnorm == 0.0:                          # R15: b = 0 -> x = 0, 0 iterations
        stats.update(converged=True, true_res=0.0)
        return np.zeros_like(b), stats
    rnd = (lambda v: v) if sloppy is None else (lambda v: v.astype(sloppy).astype(np.complex128))
    x_hi = np.zeros_like(b) if x0 is None else x0.copy()
    r_hi = b - apply_A(x_hi)                  # r0 = b - A x0 (displaced line)
    x_lo = np.zeros_like(b)
    r_lo = rnd(r_hi)
    rnorm = np.sqrt(rdot(r_lo, r_lo))
    maxr = rnorm
    k = 0
    if rnorm <= tol * bnorm:
        stats["converged"] = True
    else:
        z = precond(r_lo) if precond is not None else r_lo.copy()   # z0 = M^-1 r0
        p = z.copy()                                                 # p0 = z0
        rz = rdot(r_lo, z)
    while not stats["converged"] and k < max_iter:
        Ap = rnd(apply_A(p))
        pAp = rdot(p, Ap)
        if not pAp > 0.0:
            stats["breakdown"] = True
            break
        alpha = rz / pAp                      # alpha_k = <r_k,z_k>/<p_k,A p_k>
        x_lo = rnd(x_lo + alpha * p)          # x_{k+1} = x_k + alpha_k p_k
        r_lo = rnd(r_lo - alpha * Ap)         # r_{k+1} = r_k - alpha_k A p_k
        rnorm = np.sqrt(rdot(r_lo, r_lo))
        k += 1
        if history is not None:
            history.append(rnorm / bnorm)
        replaced = False
        if rnorm <= tol * bnorm or (sloppy is not None and rnorm < delta * maxr):
            # R17 residual replacement / R15 confirmation with the true residual
            x_hi = x_hi + x_lo
            x_lo = np.zeros_like(b)
            r_hi = b - apply_A(x_hi)
            r_lo = rnd(r_hi)
            rnorm = np.sqrt(rdot(r_hi, r_hi))
            maxr = rnorm
            stats["reliable_updates"] += 1
            replaced = True
            if rnorm <= tol * bnorm:
                stats["converged"] = True
                break
        maxr = max(maxr, rnorm)
        z = precond(r_lo) if precond is not None else r_lo.copy()   # z_{k+1} = M^-1 r_{k+1}
        rz_new = rdot(r_lo, z)
        if replaced:
            beta = rz_new / rz                # R16: Alg. 1's ratio right after a replacement (r_k is no longer the predecessor)
        else:
            # eq. 18: <z_{k+1}, r_{k+1} - r_k>/<z_k, r_k>, and r_{k+1} - r_k = -alpha_k A p_k exactly (the line above)
            beta = -alpha * rdot(z, Ap) / rz
        p = rnd(z + beta * p)                 # p_{k+1} = z_{k+1} + beta_k p_k
        rz = rz_new
    x = x_hi + x_lo
    stats["iters"] = k
    rt = b - apply_A(x)
    stats["true_res"] = float(np.sqrt(rdot(rt, rt)) / bnorm)
    return x, stats
