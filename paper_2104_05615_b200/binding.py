"""Thin ctypes binding of libmspcg (include/mspcg.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used here only to own device
memory (torch tensors) and to name the current CUDA stream.  There is no CPU fallback: if the library is missing
or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("MSPCG_LIB", os.path.join(HERE, "libmspcg.so"))   # MSPCG_LIB: an alternative build (kernel experiments)

F64, F32, F16 = 8, 4, 2
LAYOUT_ABI, LAYOUT_NATIVE = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ENOGAUGE, ENOCONV, EBREAKDOWN, ENOWORKSPACE = 0, -1, -2, -3, -4, -5, -6, -7

SYMBOLS = [
    "mspcg_create", "mspcg_destroy", "mspcg_last_error", "mspcg_geometry", "mspcg_get_matrix",
    "mspcg_workspace_bytes", "mspcg_set_workspace", "mspcg_load_gauge", "mspcg_vec_bytes", "mspcg_pack",
    "mspcg_unpack", "mspcg_apply_MdagM", "mspcg_apply_precond", "mspcg_apply_MdagM_host",
    "mspcg_apply_precond_host", "mspcg_apply_A_block", "mspcg_set_reduced_ls", "mspcg_solve", "mspcg_launch_count",
    "mspcg_timing", "mspcg_timing_read", "mspcg_update_T", "mspcg_train_eval", "mspcg_train_T",
    "mspcg_prepare_source", "mspcg_reconstruct_odd", "mspcg_apply_full", "mspcg_apply_M5inv", "mspcg_residual", "mspcg_set_block_group", "mspcg_tile_check", "mspcg_apply_MdagM_host32", "mspcg_apply_precond_host32",
    "mspcg_dot2_noalloc", "mspcg_dot2_noalloc_max_reals", "mspcg_noalloc_last_error",
    "mspcg_fixed_pack", "mspcg_fixed_unpack", "mspcg_set_fixed_storage",
]


class SolveParams(C.Structure):
    _fields_ = [("tol", C.c_double), ("max_iter", C.c_int), ("use_precond", C.c_int), ("n_inner", C.c_int),
                ("sloppy_prec", C.c_int), ("delta", C.c_double), ("use_reduced_ls", C.c_int),
                ("history_len", C.c_int), ("history", C.POINTER(C.c_double))]


class SolveStats(C.Structure):
    _fields_ = [("iters", C.c_int), ("reliable_updates", C.c_int), ("converged", C.c_int), ("breakdown", C.c_int),
                ("inner_applies", C.c_long), ("outer_applies", C.c_long), ("true_res", C.c_double),
                ("seconds", C.c_double)]


_lib = None


def load_library():
    """dlopen libmspcg.so and declare the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2104_05615_b200.build` (no CPU fallback exists)")
    L = C.CDLL(LIB_PATH)
    vp, dp, i, d = C.c_void_p, C.POINTER(C.c_double), C.c_int, C.c_double
    L.mspcg_create.argtypes = [C.POINTER(vp), i, i, i, i, i, d, d, d, d, i, i, i, i]
    L.mspcg_destroy.argtypes = [vp]
    L.mspcg_last_error.argtypes = [vp]
    L.mspcg_last_error.restype = C.c_char_p
    L.mspcg_geometry.argtypes = [vp, C.POINTER(C.c_long)]
    L.mspcg_get_matrix.argtypes = [vp, i, dp]
    L.mspcg_workspace_bytes.argtypes = [vp, i, i, i, C.POINTER(C.c_size_t)]
    L.mspcg_set_workspace.argtypes = [vp, vp, C.c_size_t, vp]
    L.mspcg_load_gauge.argtypes = [vp, vp, i, vp]
    L.mspcg_vec_bytes.argtypes = [vp, i]
    L.mspcg_vec_bytes.restype = C.c_size_t
    L.mspcg_pack.argtypes = [vp, vp, vp, i, vp]
    L.mspcg_unpack.argtypes = [vp, vp, vp, i, vp]
    L.mspcg_apply_MdagM.argtypes = [vp, vp, vp, i, i, vp]
    L.mspcg_apply_M5inv.argtypes = [vp, vp, vp, i, vp]
    L.mspcg_apply_precond.argtypes = [vp, vp, vp, i, i, i, i, vp]
    L.mspcg_apply_MdagM_host.argtypes = [vp, vp, vp, i]
    L.mspcg_apply_precond_host.argtypes = [vp, vp, vp, i, i, i]
    L.mspcg_apply_MdagM_host32.argtypes = [vp, vp, vp, i]
    L.mspcg_apply_precond_host32.argtypes = [vp, vp, vp, i, i, i]
    L.mspcg_apply_A_block.argtypes = [vp, vp, vp, i, i, vp]
    L.mspcg_prepare_source.argtypes = [vp, vp, vp, vp, vp, vp]
    L.mspcg_reconstruct_odd.argtypes = [vp, vp, vp, vp, vp]
    L.mspcg_apply_full.argtypes = [vp, vp, vp, vp, vp, vp]
    L.mspcg_residual.argtypes = [vp, vp, vp, vp, i, dp, vp]
    L.mspcg_set_block_group.argtypes = [vp, i]
    L.mspcg_tile_check.argtypes = [vp, dp]
    L.mspcg_set_reduced_ls.argtypes = [vp, i, dp, d]
    L.mspcg_solve.argtypes = [vp, vp, vp, C.POINTER(SolveParams), C.POINTER(SolveStats), vp]
    L.mspcg_launch_count.argtypes = [vp]
    L.mspcg_launch_count.restype = C.c_long
    L.mspcg_update_T.argtypes = [vp, dp, d, vp]
    L.mspcg_train_eval.argtypes = [vp, vp, i, i, dp, dp, vp]
    L.mspcg_train_T.argtypes = [vp, vp, i, i, i, d, dp, dp, vp]
    L.mspcg_timing.argtypes = [vp, i]
    L.mspcg_timing_read.argtypes = [vp, dp, C.POINTER(C.c_long)]
    L.mspcg_fixed_pack.argtypes = [vp, vp, vp, vp, i, vp]
    L.mspcg_fixed_unpack.argtypes = [vp, vp, vp, vp, i, vp]
    L.mspcg_set_fixed_storage.argtypes = [vp, i]
    L.mspcg_dot2_noalloc.argtypes = [vp, vp, vp, C.c_long, vp, vp]
    L.mspcg_dot2_noalloc_max_reals.argtypes = []
    L.mspcg_dot2_noalloc_max_reals.restype = C.c_long
    L.mspcg_noalloc_last_error.argtypes = []
    L.mspcg_noalloc_last_error.restype = C.c_char_p
    _lib = L
    return L


class MspcgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mspcg error {code}: {msg}")
        self.code = code


_TORCH_DTYPE = None


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: libmspcg has no CPU path")
    return torch


def _dtype(prec):
    torch = _torch()
    return {F64: torch.float64, F32: torch.float32, F16: torch.float16}[prec]


def dot2_noalloc(a, b, c, out):
    """mspcg_dot2_noalloc: out[0] = <a,b>, out[1] = <a,c> (c may be None) over all reals of the fp64 CUDA tensors a, b, c, into the
    caller's 2-element fp64 CUDA tensor `out`, on torch's current stream.  Allocates nothing (the library's static scratch array)."""
    torch = _torch()
    lib = load_library()
    for t in (a, b, out) + ((c,) if c is not None else ()):
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise ValueError("dot2_noalloc wants contiguous fp64 CUDA tensors")
    if b.numel() != a.numel() or (c is not None and c.numel() != a.numel()) or out.numel() < 2:
        raise ValueError("dot2_noalloc: size mismatch")
    rc = lib.mspcg_dot2_noalloc(C.c_void_p(a.data_ptr()), C.c_void_p(b.data_ptr()), C.c_void_p(c.data_ptr() if c is not None else None),
                                a.numel(), C.c_void_p(out.data_ptr()), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != 0:
        raise MspcgError(rc, lib.mspcg_noalloc_last_error().decode())
    return out


class Mspcg:
    """One mspcg_ctx.  Tensors passed in and out are torch CUDA tensors; the workspace is a torch uint8 tensor."""

    def __init__(self, dims, Ls, b, c, M5, mf, block=None):
        self.lib = load_library()
        self.dims = tuple(int(x) for x in dims)
        self.Ls = int(Ls)
        self.block = tuple(int(x) for x in (block if block is not None else dims))
        h = C.c_void_p()
        rc = self.lib.mspcg_create(C.byref(h), *self.dims, self.Ls, b, c, M5, mf, *self.block)
        if rc != OK:
            raise MspcgError(rc, "mspcg_create rejected the parameters")
        self.h = h
        self.vh = int(np.prod(self.dims)) // 2
        self.nreal = self.Ls * self.vh * 24
        self.workspace = None
        self.outer_prec = self.inner_prec = None

    def close(self):
        if getattr(self, "h", None):
            self.lib.mspcg_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, allow=()):
        if rc != OK and rc not in allow:
            raise MspcgError(rc, self.lib.mspcg_last_error(self.h).decode())
        return rc

    # ---- host-only queries -------------------------------------------------------------------------------------
    def geometry(self):
        out = (C.c_long * 5)()
        self._check(self.lib.mspcg_geometry(self.h, out))
        return dict(nblk=out[0], nE0=out[1], nE2=out[2], nO1=out[3], vh=out[4])

    def matrix(self, which):
        out = np.empty((self.Ls, self.Ls))
        self._check(self.lib.mspcg_get_matrix(self.h, {"m5": 0, "mphi": 1, "m5inv": 2}[which],
                                              out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def workspace_bytes(self, outer_prec=F32, inner_prec=F16, recon=18):
        n = C.c_size_t()
        self._check(self.lib.mspcg_workspace_bytes(self.h, outer_prec, inner_prec, recon, C.byref(n)))
        self.outer_prec, self.inner_prec = outer_prec, inner_prec
        return n.value

    def set_reduced_ls(self, Ls_hat, T_abi, mu):
        """Reduced-Ls preconditioner: T_abi = float64 [4*Ls_hat][4*Ls][re,im]; call before configure()."""
        T = np.ascontiguousarray(T_abi, dtype=np.float64).reshape(-1)
        assert T.size == 4 * int(Ls_hat) * 4 * self.Ls * 2
        self._check(self.lib.mspcg_set_reduced_ls(self.h, int(Ls_hat), T.ctypes.data_as(C.POINTER(C.c_double)), float(mu)))
        self.Ls_hat = int(Ls_hat)

    def update_T(self, T_abi, mu):
        T = np.ascontiguousarray(T_abi, dtype=np.float64).reshape(-1)
        self._check(self.lib.mspcg_update_T(self.h, T.ctypes.data_as(C.POINTER(C.c_double)), float(mu), self._stream()))

    def train_eval(self, vs, n_inner, want_grad=True):
        """chi2 of eq. 22 (and its gradient, layout of T_abi) for the current T; vs: torch fp64 CUDA tensor [nvec * nreal]."""
        nvec = vs.numel() // self.nreal
        chi2 = C.c_double()
        G = np.zeros(4 * self.Ls_hat * 4 * self.Ls * 2)
        gp = G.ctypes.data_as(C.POINTER(C.c_double)) if want_grad else None
        self._check(self.lib.mspcg_train_eval(self.h, C.c_void_p(vs.data_ptr()), nvec, int(n_inner), C.byref(chi2), gp, self._stream()))
        return chi2.value, (G if want_grad else None)

    def train_T(self, vs, n_inner, n_steps, momentum=0.0):
        nvec = vs.numel() // self.nreal
        T = np.zeros(4 * self.Ls_hat * 4 * self.Ls * 2)
        hist = np.zeros(n_steps + 1)
        self._check(self.lib.mspcg_train_T(self.h, C.c_void_p(vs.data_ptr()), nvec, int(n_inner), int(n_steps), float(momentum),
                                           T.ctypes.data_as(C.POINTER(C.c_double)), hist.ctypes.data_as(C.POINTER(C.c_double)), self._stream()))
        return T, hist

    # ---- device set-up -----------------------------------------------------------------------------------------
    def _stream(self):
        return C.c_void_p(_torch().cuda.current_stream().cuda_stream)

    def configure(self, outer_prec=F32, inner_prec=F16, recon=18):
        torch = _torch()
        n = self.workspace_bytes(outer_prec, inner_prec, recon)
        self.workspace = torch.empty(n + 256, dtype=torch.uint8, device="cuda")
        ptr = (self.workspace.data_ptr() + 255) & ~255
        self._check(self.lib.mspcg_set_workspace(self.h, C.c_void_p(ptr), n, self._stream()))
        return n

    def load_gauge(self, U_abi, t_boundary=-1):
        torch = _torch()
        U = torch.as_tensor(np.ascontiguousarray(U_abi, dtype=np.float64)).cuda() if not hasattr(U_abi, "data_ptr") else U_abi
        assert U.numel() == 4 * 2 * self.vh * 18 and U.dtype == torch.float64 and U.is_contiguous()
        self._check(self.lib.mspcg_load_gauge(self.h, C.c_void_p(U.data_ptr()), int(t_boundary), self._stream()))
        torch.cuda.current_stream().synchronize()  # U may be a temporary

    # ---- vectors -----------------------------------------------------------------------------------------------
    def new_native(self, prec):
        torch = _torch()
        return torch.empty(self.nreal, dtype=_dtype(prec), device="cuda")

    def pack(self, abi, prec, out=None):
        torch = _torch()
        assert abi.dtype == torch.float64 and abi.numel() == self.nreal and abi.is_contiguous()
        out = self.new_native(prec) if out is None else out
        self._check(self.lib.mspcg_pack(self.h, C.c_void_p(abi.data_ptr()), C.c_void_p(out.data_ptr()), prec, self._stream()))
        return out

    def unpack(self, nat, prec, out=None):
        torch = _torch()
        out = torch.empty(self.nreal, dtype=torch.float64, device="cuda") if out is None else out
        self._check(self.lib.mspcg_unpack(self.h, C.c_void_p(nat.data_ptr()), C.c_void_p(out.data_ptr()), prec, self._stream()))
        return out

    # ---- the hot path ------------------------------------------------------------------------------------------
    def apply_MdagM(self, v, prec=F64, layout=LAYOUT_ABI, out=None):
        torch = _torch()
        out = torch.empty_like(v) if out is None else out
        self._check(self.lib.mspcg_apply_MdagM(self.h, C.c_void_p(v.data_ptr()), C.c_void_p(out.data_ptr()), prec, layout, self._stream()))
        return out

    def apply_M5inv(self, v_native_f16, dagger=False, out=None):
        torch = _torch()
        out = torch.empty_like(v_native_f16) if out is None else out
        self._check(self.lib.mspcg_apply_M5inv(self.h, C.c_void_p(v_native_f16.data_ptr()), C.c_void_p(out.data_ptr()), int(bool(dagger)), self._stream()))
        return out

    def apply_precond(self, r, n_inner, io_prec=F64, layout=LAYOUT_ABI, out=None, use_reduced=0):
        torch = _torch()
        out = torch.empty_like(r) if out is None else out
        self._check(self.lib.mspcg_apply_precond(self.h, C.c_void_p(r.data_ptr()), C.c_void_p(out.data_ptr()), io_prec, layout,
                                                 int(n_inner), int(use_reduced), self._stream()))
        return out

    def apply_A_block(self, v_abi, block, prec=None):
        torch = _torch()
        out = torch.empty_like(v_abi)
        self._check(self.lib.mspcg_apply_A_block(self.h, C.c_void_p(v_abi.data_ptr()), C.c_void_p(out.data_ptr()), int(block),
                                                 prec if prec is not None else self.inner_prec, self._stream()))
        return out

    def prepare_source(self, phi_e_abi, phi_o_abi):
        """(phihat_e, D^dag phihat_e) of PAPER.md:97 eq. 6 and PAPER.md:117 eq. 9; fp64 ABI device tensors."""
        torch = _torch()
        hat, rhs = torch.empty_like(phi_e_abi), torch.empty_like(phi_e_abi)
        self._check(self.lib.mspcg_prepare_source(self.h, C.c_void_p(phi_e_abi.data_ptr()), C.c_void_p(phi_o_abi.data_ptr()),
                                                  C.c_void_p(hat.data_ptr()), C.c_void_p(rhs.data_ptr()), self._stream()))
        return hat, rhs

    def reconstruct_odd(self, psi_e_abi, phi_o_abi):
        torch = _torch()
        out = torch.empty_like(phi_o_abi)
        self._check(self.lib.mspcg_reconstruct_odd(self.h, C.c_void_p(psi_e_abi.data_ptr()), C.c_void_p(phi_o_abi.data_ptr()),
                                                   C.c_void_p(out.data_ptr()), self._stream()))
        return out

    def apply_full(self, psi_e_abi, psi_o_abi):
        torch = _torch()
        oe, oo = torch.empty_like(psi_e_abi), torch.empty_like(psi_o_abi)
        self._check(self.lib.mspcg_apply_full(self.h, C.c_void_p(psi_e_abi.data_ptr()), C.c_void_p(psi_o_abi.data_ptr()),
                                              C.c_void_p(oe.data_ptr()), C.c_void_p(oo.data_ptr()), self._stream()))
        return oe, oo

    def tile_check(self):
        """Host-only consistency check of the tile tables of the fp16 tile kernel (mspcg_tile_check); raises on failure."""
        out = np.zeros(8)
        self._check(self.lib.mspcg_tile_check(self.h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return dict(tiles_k2=int(out[1]), tiles_k4=int(out[2]), tiles_k3k5=int(out[3]), tiles_k3_halo=int(out[4]),
                    inputs_per_output_k4=out[5], inputs_per_output_k3k5=out[6], inputs_per_output_full=out[7])

    def set_block_group(self, blocks_per_group):
        """L2-resident groups of Dirichlet blocks for the preconditioner (mspcg_set_block_group); 0 = all blocks at once."""
        self._check(self.lib.mspcg_set_block_group(self.h, int(blocks_per_group)))

    def set_fixed_storage(self, bits):
        """fp32 inner CG vectors pass through the 8- / 16-bit fixed-point store of eq. 17 (mspcg_set_fixed_storage); 0 = off."""
        self._check(self.lib.mspcg_set_fixed_storage(self.h, int(bits)))

    def fixed_pack(self, v_abi, bits):
        """ABI vector -> (integers [Ls*V/2*24] int8 / int16, scales [Ls*V/2] float32) in the fixed-point format of eq. 17 (mspcg_fixed_pack)."""
        torch = _torch()
        n = v_abi.numel() // 24
        q = torch.empty(n * 24, dtype=torch.int8 if bits == 8 else torch.int16, device="cuda")
        sc = torch.empty(n, dtype=torch.float32, device="cuda")
        self._check(self.lib.mspcg_fixed_pack(self.h, C.c_void_p(v_abi.data_ptr()), C.c_void_p(q.data_ptr()), C.c_void_p(sc.data_ptr()), int(bits), self._stream()))
        return q, sc

    def fixed_unpack(self, q, sc, bits):
        torch = _torch()
        out = torch.empty(q.numel(), dtype=torch.float64, device="cuda")
        self._check(self.lib.mspcg_fixed_unpack(self.h, C.c_void_p(q.data_ptr()), C.c_void_p(sc.data_ptr()), C.c_void_p(out.data_ptr()), int(bits), self._stream()))
        return out

    def residual(self, b_abi, x_abi, normalise=False):
        """r = b - D^dag D x in fp64 (mspcg_residual), optionally divided by its norm; returns (r, |b - D^dag D x|)."""
        torch = _torch()
        r = torch.empty_like(b_abi)
        rn = C.c_double()
        self._check(self.lib.mspcg_residual(self.h, C.c_void_p(b_abi.data_ptr()), C.c_void_p(x_abi.data_ptr()), C.c_void_p(r.data_ptr()),
                                            int(bool(normalise)), C.byref(rn), self._stream()))
        return r, rn.value

    def apply_MdagM_host(self, v_host, out_host, prec=F64):
        self._check(self.lib.mspcg_apply_MdagM_host(self.h, C.c_void_p(v_host.data_ptr()), C.c_void_p(out_host.data_ptr()), prec))
        return out_host

    def apply_MdagM_host32(self, v_host, out_host, prec=F32):
        """float32 host tensors in the ABI layout (mspcg_apply_MdagM_host32)."""
        self._check(self.lib.mspcg_apply_MdagM_host32(self.h, C.c_void_p(v_host.data_ptr()), C.c_void_p(out_host.data_ptr()), prec))
        return out_host

    def apply_precond_host32(self, r_host, z_host, n_inner, io_prec=F32, use_reduced=0):
        self._check(self.lib.mspcg_apply_precond_host32(self.h, C.c_void_p(r_host.data_ptr()), C.c_void_p(z_host.data_ptr()), io_prec,
                                                        int(n_inner), int(use_reduced)))
        return z_host

    def apply_precond_host(self, r_host, z_host, n_inner, io_prec=F64, use_reduced=0):
        self._check(self.lib.mspcg_apply_precond_host(self.h, C.c_void_p(r_host.data_ptr()), C.c_void_p(z_host.data_ptr()), io_prec,
                                                      int(n_inner), int(use_reduced)))
        return z_host

    def solve(self, b_abi, x0_abi=None, tol=1e-10, max_iter=100000, use_precond=False, n_inner=6, sloppy_prec=F64,
              delta=0.1, use_reduced_ls=False, history_len=0):
        torch = _torch()
        x = torch.zeros_like(b_abi) if x0_abi is None else x0_abi.clone()
        hist = np.zeros(max(history_len, 1))
        prm = SolveParams(tol, int(max_iter), int(use_precond), int(n_inner), int(sloppy_prec), delta, int(use_reduced_ls),
                          int(history_len), hist.ctypes.data_as(C.POINTER(C.c_double)))
        st = SolveStats()
        rc = self.lib.mspcg_solve(self.h, C.c_void_p(b_abi.data_ptr()), C.c_void_p(x.data_ptr()), C.byref(prm), C.byref(st),
                                  self._stream())
        self._check(rc, allow=(ENOCONV, EBREAKDOWN))
        stats = {k: getattr(st, k) for k, _ in SolveStats._fields_}
        stats["rc"] = rc
        stats["history"] = hist[:min(history_len, st.iters)].copy()
        return x, stats

    def launch_count(self):
        return int(self.lib.mspcg_launch_count(self.h))

    TIMING_CLASSES = ["full.mphi", "full.hop_k2k4", "full.hop_k3", "full.hop_k5", "full.blas",
                      "blk.mphi", "blk.hop_k2k4", "blk.hop_k3", "blk.hop_k5", "blk.blas"]

    def timing(self, enable):
        self._check(self.lib.mspcg_timing(self.h, int(bool(enable))))

    def timing_read(self):
        ms = (C.c_double * 10)()
        n = (C.c_long * 10)()
        self._check(self.lib.mspcg_timing_read(self.h, ms, n))
        return {k: dict(ms=ms[j], launches=n[j]) for j, k in enumerate(self.TIMING_CLASSES)}
