"""ORACLE -- test infrastructure only (see oracle/mdwf.py header).  ABI-level entry points.

These functions mirror the five C-ABI calls of include/mspcg.h on ABI-layout numpy arrays, so
tests can hand the very same inputs to the oracle and to the CUDA library.  Nothing outside
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline/--impl reference legs may import this.
"""
from __future__ import annotations

import numpy as np

from . import mdwf, solvers


class Oracle:
    """Holds (lattice, Moebius parameters, folded links, block partition) like an mspcg_ctx."""

    def __init__(self, dims, Ls, b, c, M5, mf, block=None):
        self.dims = tuple(int(d) for d in dims)
        if any(d % 2 for d in self.dims):
            raise ValueError("all lattice extents must be even (R5)")
        self.mob = mdwf.Mobius(Ls, b, c, M5, mf)
        self.Ls = int(Ls)
        self.block = tuple(block) if block is not None else self.dims
        self.U = None
        self._pre = {}

    def load_gauge(self, U_abi, t_boundary=-1):
        self.U = mdwf.fold_t_boundary(mdwf.unpack_gauge_abi(U_abi, self.dims), t_boundary)
        self._pre = {}

    # -- helpers ---------------------------------------------------------
    def unpack(self, v_abi):
        return mdwf.unpack_spinor_abi(v_abi, self.dims, self.Ls, 0)

    def pack(self, v):
        return mdwf.pack_spinor_abi(v, self.dims, 0)

    def precond_obj(self, variant="PAD"):
        if variant not in self._pre:
            self._pre[variant] = solvers.BlockPrecond(self.mob, self.U, self.dims, self.block, variant)
        return self._pre[variant]

    # -- the five calls ----------------------------------------------------
    def apply_MdagM(self, in_abi):
        return self.pack(mdwf.MdagM(self.mob, self.U, self.unpack(in_abi)))

    def apply_D(self, in_abi, dagger=False):
        f = mdwf.D_eo_dag if dagger else mdwf.D_eo
        return self.pack(f(self.mob, self.U, self.unpack(in_abi)))

    # -- full 4-step solve (eq. 4-6, eq. 9) ----------------------------
    def unpack_odd(self, v_abi):
        return mdwf.unpack_spinor_abi(v_abi, self.dims, self.Ls, 1)

    def pack_odd(self, v):
        return mdwf.pack_spinor_abi(v, self.dims, 1)

    def prepare_source(self, phi_e_abi, phi_o_abi):
        """(phihat_e of eq. 6, D^dag phihat_e of eq. 9), both even-parity ABI vectors."""
        pe, po = self.unpack(phi_e_abi), self.unpack_odd(phi_o_abi)
        hat = mdwf.prepare_source(self.mob, self.U, pe, po)
        return self.pack(hat), self.pack(mdwf.D_eo_dag(self.mob, self.U, hat))

    def reconstruct_odd(self, psi_e_abi, phi_o_abi):
        return self.pack_odd(mdwf.reconstruct_odd(self.mob, self.U, self.unpack(psi_e_abi), self.unpack_odd(phi_o_abi)))

    def apply_full(self, psi_e_abi, psi_o_abi):
        """The unpreconditioned 2x2 operator of eq. (4) -> (even part, odd part)."""
        out = mdwf.D_dw(self.mob, self.U, self.unpack(psi_e_abi) + self.unpack_odd(psi_o_abi))
        return self.pack(out), self.pack_odd(out)

    def apply_precond(self, r_abi, n_inner, variant="PAD", blocks=None):
        return self.pack(self.precond_obj(variant)(self.unpack(r_abi), n_inner, blocks))

    def apply_A_block(self, v_abi, block_index, variant="PAD"):
        pre = self.precond_obj(variant)
        return self.pack(pre.apply_A_block(pre.origins[block_index], self.unpack(v_abi)))

    def solve(self, b_abi, tol=1e-10, max_iter=100000, use_precond=False, n_inner=6,
              sloppy=None, delta=0.1, x0_abi=None, history=None, variant="PAD"):
        A = lambda v: mdwf.MdagM(self.mob, self.U, v)
        pre = None
        if use_precond:
            P = self.precond_obj(variant)
            pre = lambda r: P(r, n_inner)
        x0 = None if x0_abi is None else self.unpack(x0_abi)
        x, stats = solvers.pcg(A, self.unpack(b_abi), pre, tol, max_iter, x0, sloppy, delta, history)
        if use_precond:
            stats["inner_applies"] = self.precond_obj(variant).napply
        return self.pack(x), stats
