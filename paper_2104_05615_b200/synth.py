"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests/bench.

This module holds NONE of the method's arithmetic (no Dirac operator, no
preconditioner, no CG): only random-number generation, the SU(3) exponential
map used to make links, and pure index permutations into the C-ABI layouts of
include/mspcg.h.  Both the oracle (oracle/) and the CUDA library are fed the
SAME ABI-layout arrays produced here; neither imports the other.

Input recipe: the paper measures
on RBC/UKQCD and CalLat gauge ensembles which are not
available; seeded synthetic SU(3) fields with the paper's shapes stand in.

  links : rng = numpy.random.default_rng(seed); for every link, in the order
          [mu][t][z][y][x], G = N(0,1)+iN(0,1) (3x3), H = (G+G^dag)/2 - tr/3,
          U = V exp(i*eps*lambda) V^dag from eigh(H).  eps is the "roughness".
  source: real and imaginary parts iid N(0,1) on even sites in ABI order.

ABI layouts (see include/mspcg.h):
  gauge  U_abi[mu][parity][x_cb][row][col][re,im]  float64
  spinor psi_abi[s][x_cb][spin][colour][re,im]      float64 (even parity)
  x_cb = lex(x,y,z,t)/2 with lex = x + Lx*(y + Ly*(z + Lz*t)), parity=(x+y+z+t)%2.
"""
from __future__ import annotations

import numpy as np


def lattice_volume(dims):
    Lx, Ly, Lz, Lt = dims
    return Lx * Ly * Lz * Lt


def parity_mask(dims):
    """Boolean array [t,z,y,x]: True on odd sites ((x+y+z+t)%2==1), eq. 3."""
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return ((x + y + z + t) & 1).astype(bool)


def checkerboard_index(dims):
    """lex indices (into the flattened [t,z,y,x] array) of even and odd sites, in x_cb order."""
    odd = parity_mask(dims).reshape(-1)
    lex = np.arange(odd.size)
    return lex[~odd], lex[odd]


def random_su3_links(dims, eps, seed, batch=1 << 16):
    """Natural-order links U[mu,t,z,y,x,3,3] complex128, U = exp(i*eps*H), H random traceless Hermitian."""
    Lx, Ly, Lz, Lt = dims
    n = 4 * Lt * Lz * Ly * Lx
    rng = np.random.default_rng(seed)
    out = np.empty((n, 3, 3), dtype=np.complex128)
    for lo in range(0, n, batch):
        hi = min(n, lo + batch)
        g = rng.standard_normal((hi - lo, 3, 3, 2))
        G = g[..., 0] + 1j * g[..., 1]
        H = 0.5 * (G + np.conj(np.swapaxes(G, -1, -2)))
        tr = np.trace(H, axis1=-2, axis2=-1) / 3.0
        H = H - tr[:, None, None] * np.eye(3)
        lam, V = np.linalg.eigh(H)
        ph = np.exp(1j * eps * lam)
        out[lo:hi] = np.einsum("nab,nb,ncb->nac", V, ph, np.conj(V))
    return out.reshape(4, Lt, Lz, Ly, Lx, 3, 3)


def unit_links(dims):
    Lx, Ly, Lz, Lt = dims
    U = np.zeros((4, Lt, Lz, Ly, Lx, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1.0
    return U


def random_su3_field(dims, seed):
    """One Haar-ish SU(3) matrix per 4D site, g[t,z,y,x,3,3] (for gauge-covariance tests)."""
    Lx, Ly, Lz, Lt = dims
    rng = np.random.default_rng(seed)
    n = Lt * Lz * Ly * Lx
    g = rng.standard_normal((n, 3, 3, 2))
    G = g[..., 0] + 1j * g[..., 1]
    Q, R = np.linalg.qr(G)
    d = np.diagonal(R, axis1=-2, axis2=-1)
    Q = Q * (d / np.abs(d))[:, None, :]
    det = np.linalg.det(Q)
    Q = Q * (np.conj(det) ** (1.0 / 3.0))[:, None, None]
    return Q.reshape(Lt, Lz, Ly, Lx, 3, 3)


def gauge_natural_to_abi(U, dims):
    """Pure permutation: U[mu,t,z,y,x,3,3] complex -> U_abi[mu][parity][x_cb][3][3][2] float64."""
    ev, od = checkerboard_index(dims)
    Uf = U.reshape(4, -1, 3, 3)
    out = np.empty((4, 2, ev.size, 3, 3, 2), dtype=np.float64)
    for p, idx in enumerate((ev, od)):
        out[:, p, :, :, :, 0] = Uf[:, idx].real
        out[:, p, :, :, :, 1] = Uf[:, idx].imag
    return out


def gauge_abi_to_natural(U_abi, dims):
    Lx, Ly, Lz, Lt = dims
    ev, od = checkerboard_index(dims)
    Uf = np.empty((4, Lx * Ly * Lz * Lt, 3, 3), dtype=np.complex128)
    for p, idx in enumerate((ev, od)):
        Uf[:, idx] = U_abi[:, p, :, :, :, 0] + 1j * U_abi[:, p, :, :, :, 1]
    return Uf.reshape(4, Lt, Lz, Ly, Lx, 3, 3)


def gaussian_spinor_abi(dims, Ls, seed):
    """psi_abi[s][x_cb][4][3][2] float64, iid N(0,1), even-parity half lattice."""
    rng = np.random.default_rng(seed)
    return rng.standard_normal((Ls, lattice_volume(dims) // 2, 4, 3, 2))


def gauge_transform_links(U, g):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag (natural order); used only by covariance tests."""
    out = np.empty_like(U)
    for mu in range(4):
        axis = 3 - mu  # g is [t,z,y,x,...]
        g_fwd = np.roll(g, -1, axis=axis)
        out[mu] = np.einsum("...ab,...bc,...dc->...ad", g, U[mu], np.conj(g_fwd))
    return out


def gauge_transform_spinor_abi(psi_abi, g, dims, parity=0):
    """psi'(x) = g(x) psi(x) on the given parity, ABI layout in and out."""
    ev, od = checkerboard_index(dims)
    idx = ev if parity == 0 else od
    gf = g.reshape(-1, 3, 3)[idx]
    psi = psi_abi[..., 0] + 1j * psi_abi[..., 1]
    out = np.einsum("xab,sxib->sxia", gf, psi)
    return np.stack([out.real, out.imag], axis=-1)


# ---------------------------------------------------------------------------
# The five BASELINE.json configurations (C1..C5) + reduced variants used by tests.
# ---------------------------------------------------------------------------
MOBIUS = dict(b=1.5, c=0.5, M5=1.8)

CONFIGS = {
    "C1": dict(dims=(4, 4, 4, 4), Ls=8, mf=0.01, eps=0.3, gauge_seed=0, src_seed=1,
               block=(2, 2, 2, 2), n_inner=6, **MOBIUS),
    "C2": dict(dims=(16, 16, 16, 32), Ls=16, mf=0.01, eps=0.2, gauge_seed=12, src_seed=22,
               block=(8, 8, 8, 8), n_inner=6, **MOBIUS),
    "C3": dict(dims=(24, 24, 24, 64), Ls=16, mf=0.002, eps=0.1, gauge_seed=13, src_seed=2,
               block=(12, 12, 12, 16), n_inner=5, **MOBIUS),
    "C4": dict(dims=(32, 32, 32, 64), Ls=12, mf=0.005, eps=0.15, gauge_seed=14, src_seed=24,
               block=(16, 16, 16, 32), n_inner=6, Ls_hat=6, **MOBIUS),
    "C5": dict(dims=(48, 48, 48, 96), Ls=12, mf=0.001, eps=0.1, gauge_seed=15, src_seed=25,
               block=(8, 8, 8, 8), n_inner=6, **MOBIUS),
    # reduced C3 (SURVEY 8(d) CPU baseline plan): same parameters on a lattice the CPU oracle solves in minutes
    "C3p": dict(dims=(12, 12, 12, 24), Ls=8, mf=0.002, eps=0.1, gauge_seed=13, src_seed=2,
                block=(6, 6, 6, 12), n_inner=5, **MOBIUS),
}
