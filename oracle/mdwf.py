"""ORACLE (test infrastructure only) -- Moebius domain-wall operators written from the paper.

This file is part of the CPU oracle for arXiv 2104.05615.  It is plain
numpy in complex128/float64, unfused, unblocked, and shares NO code with the CUDA
path in paper_2104_05615_b200/.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import it.

Every function cites the passage of /root/reference/PAPER.md it follows, or the
DESIGN.md reading (R1..R20, restated from SURVEY.md 8(c)) where the paper is silent.

Internal field layout (natural order, BOTH parities present, the unused parity zero):
    psi[s, t, z, y, x, spin, colour]   complex128
    U  [mu, t, z, y, x, row, col]      complex128   (mu = 0,1,2,3 <-> x,y,z,t)
Public entry points take/return the C-ABI layouts of include/mspcg.h and unpack
them with this file's own index code.

Pins (tests/test_oracle_*.py): gamma algebra; M5inv closed form vs numpy.linalg.inv
and M5inv.M5=1; brute-force site loops of eq. 8 on a tiny lattice; free-field
momentum-space closed form (R9); Shamir limit; gamma5-hermiticity; Schur identity;
gauge covariance; dense direct solves.  No function here is "parity unpinned"
except train-related items, which live in oracle/reduced_ls.py and say so.
"""
from __future__ import annotations

import numpy as np

# ---------------------------------------------------------------------------
# R2 -- gamma matrices, chiral basis with gamma5 = diag(+1,+1,-1,-1) (paper silent).
# gamma_k = [[0, -i sigma_k], [+i sigma_k, 0]] (k = x,y,z), gamma_4 = [[0,1],[1,0]].
# ---------------------------------------------------------------------------
_s1 = np.array([[0, 1], [1, 0]], dtype=np.complex128)
_s2 = np.array([[0, -1j], [1j, 0]], dtype=np.complex128)
_s3 = np.array([[1, 0], [0, -1]], dtype=np.complex128)
_z2 = np.zeros((2, 2), dtype=np.complex128)
_i2 = np.eye(2, dtype=np.complex128)


def _offdiag(a, b):
    return np.block([[_z2, a], [b, _z2]])


GAMMA = np.stack([
    _offdiag(-1j * _s1, 1j * _s1),
    _offdiag(-1j * _s2, 1j * _s2),
    _offdiag(-1j * _s3, 1j * _s3),
    _offdiag(_i2, _i2),
])
GAMMA5 = GAMMA[0] @ GAMMA[1] @ GAMMA[2] @ GAMMA[3]
P_PLUS = 0.5 * (np.eye(4) + GAMMA5)    # selects spin 0,1
P_MINUS = 0.5 * (np.eye(4) - GAMMA5)   # selects spin 2,3

_AXIS = {0: 4, 1: 3, 2: 2, 3: 1}  # mu -> axis of psi[s,t,z,y,x,spin,colour]


# ---------------------------------------------------------------------------
# ABI <-> natural layout (own index code; include/mspcg.h states the ABI layouts)
# ---------------------------------------------------------------------------
def _cb_index(dims):
    Lx, Ly, Lz, Lt = dims
    lex = np.arange(Lx * Ly * Lz * Lt)
    x = lex % Lx
    y = (lex // Lx) % Ly
    z = (lex // (Lx * Ly)) % Lz
    t = lex // (Lx * Ly * Lz)
    par = (x + y + z + t) % 2  # PAPER.md:87 eq. 3
    return lex[par == 0], lex[par == 1]


def unpack_gauge_abi(U_abi, dims):
    """U_abi[mu][parity][x_cb][3][3][2] float64 -> U[mu,t,z,y,x,3,3] complex128."""
    Lx, Ly, Lz, Lt = dims
    ev, od = _cb_index(dims)
    U_abi = np.asarray(U_abi, dtype=np.float64).reshape(4, 2, ev.size, 3, 3, 2)
    Uf = np.empty((4, Lx * Ly * Lz * Lt, 3, 3), dtype=np.complex128)
    Uf[:, ev] = U_abi[:, 0, ..., 0] + 1j * U_abi[:, 0, ..., 1]
    Uf[:, od] = U_abi[:, 1, ..., 0] + 1j * U_abi[:, 1, ..., 1]
    return Uf.reshape(4, Lt, Lz, Ly, Lx, 3, 3)


def unpack_spinor_abi(psi_abi, dims, Ls, parity=0):
    """psi_abi[s][x_cb][4][3][2] -> psi[s,t,z,y,x,4,3] with zeros on the other parity."""
    Lx, Ly, Lz, Lt = dims
    idx = _cb_index(dims)[parity]
    a = np.asarray(psi_abi, dtype=np.float64).reshape(Ls, idx.size, 4, 3, 2)
    full = np.zeros((Ls, Lx * Ly * Lz * Lt, 4, 3), dtype=np.complex128)
    full[:, idx] = a[..., 0] + 1j * a[..., 1]
    return full.reshape(Ls, Lt, Lz, Ly, Lx, 4, 3)


def pack_spinor_abi(psi, dims, parity=0):
    Ls = psi.shape[0]
    idx = _cb_index(dims)[parity]
    f = psi.reshape(Ls, -1, 4, 3)[:, idx]
    return np.stack([f.real, f.imag], axis=-1)


def fold_t_boundary(U, t_boundary):
    """R7: antiperiodic time = multiply U_t(x,y,z,Lt-1) by -1; user passes periodic links."""
    U = U.copy()
    if t_boundary == -1:
        U[3, -1] *= -1.0
    elif t_boundary != 1:
        raise ValueError("t_boundary must be +1 or -1")
    return U


# ---------------------------------------------------------------------------
# PAPER.md:105 eq. (8) -- the Wilson hopping term D^w
#   D^w_{x,y} = sum_mu [ (1+gamma_mu) U^dag_{x-mu,mu} delta_{x-mu,y}
#                      + (1-gamma_mu) U_{x,mu}       delta_{x+mu,y} ]
# dagger=True gives D^w^dag = the same with gamma_mu -> -gamma_mu (R6).
# periodic[mu]=False applies a zero Dirichlet condition at the array boundary in
# direction mu (used for the padded box of PAPER.md:224).
# ---------------------------------------------------------------------------
def _shift(a, axis, disp, periodic):
    """b[x] = a[x + disp*e_axis]; zero fill instead of wrap when not periodic."""
    b = np.roll(a, -disp, axis=axis)
    if not periodic:
        sl = [slice(None)] * a.ndim
        sl[axis] = slice(-1, None) if disp > 0 else slice(0, 1)
        b[tuple(sl)] = 0.0
    return b


def hop(U, psi, dagger=False, periodic=(True, True, True, True)):
    sgn = -1.0 if dagger else 1.0
    out = np.zeros_like(psi)
    eye = np.eye(4)
    for mu in range(4):
        ax = _AXIS[mu]
        # (1 - gamma_mu) U_mu(x) psi(x+mu)
        fwd = np.einsum("tzyxab,stzyxib->stzyxia", U[mu], _shift(psi, ax, +1, periodic[mu]))
        out += np.einsum("ij,stzyxjc->stzyxic", eye - sgn * GAMMA[mu], fwd)
        # (1 + gamma_mu) U_mu(x-mu)^dag psi(x-mu)
        w = np.einsum("tzyxba,stzyxib->stzyxia", np.conj(U[mu]), psi)
        bwd = _shift(w, ax, -1, periodic[mu])
        out += np.einsum("ij,stzyxjc->stzyxic", eye + sgn * GAMMA[mu], bwd)
    return out


# ---------------------------------------------------------------------------
# R1/R3 -- fifth-dimension operators.  (L psi)_s = P- psi_{s+1} + P+ psi_{s-1} with
# P- psi_{Ls} = -mf P- psi_0 and P+ psi_{-1} = -mf P+ psi_{Ls-1}.
#   M5   = alpha + beta L,  alpha = b(4-M5)+1, beta = c(4-M5)-1   (eq. 4 diag blocks)
#   Mphi = -(b + c L)/2                                            (eq. 7)
# On P+ components every such operator is the real Ls x Ls matrix  a*1 + d*S_minus,
# (S_minus psi)_s = psi_{s-1}, (S_minus psi)_0 = -mf psi_{Ls-1}; on P- components its transpose.
# The dagger swaps the two (all entries real).
# ---------------------------------------------------------------------------
class Mobius:
    def __init__(self, Ls, b, c, M5, mf):
        self.Ls, self.b, self.c, self.M5, self.mf = int(Ls), float(b), float(c), float(M5), float(mf)
        self.alpha = self.b * (4.0 - self.M5) + 1.0
        self.beta = self.c * (4.0 - self.M5) - 1.0
        if self.alpha == 0.0:
            raise ValueError("alpha = b(4-M5)+1 must be non-zero")

    def s_minus(self):
        Ls = self.Ls
        S = np.zeros((Ls, Ls))
        for s in range(1, Ls):
            S[s, s - 1] = 1.0
        S[0, Ls - 1] = -self.mf
        return S

    def m5_plus(self):
        return self.alpha * np.eye(self.Ls) + self.beta * self.s_minus()

    def mphi_plus(self):
        return -0.5 * (self.b * np.eye(self.Ls) + self.c * self.s_minus())

    def m5inv_plus_closed_form(self):
        """R4: (A+^-1)[s,s'] = (-k)^((s-s') mod Ls) (1 if s>=s' else -mf) / (alpha (1 + mf (-k)^Ls)), k = beta/alpha."""
        Ls, mf = self.Ls, self.mf
        k = self.beta / self.alpha
        den = self.alpha * (1.0 + mf * (-k) ** Ls)
        A = np.empty((Ls, Ls))
        for s in range(Ls):
            for sp in range(Ls):
                A[s, sp] = (-k) ** ((s - sp) % Ls) * (1.0 if s >= sp else -mf) / den
        return A


def apply_5d(mat_plus, psi, dagger=False):
    """Apply a 4D-diagonal operator given by its P+ block `mat_plus` (P- block = transpose).

    PAPER.md:103: "M5 and Mphi are constant matrices that are diagonal in the 4D
    Euclidean space-time dimensions"; chirality structure from R3.
    """
    up = mat_plus.T if dagger else mat_plus
    dn = mat_plus if dagger else mat_plus.T
    out = np.empty_like(psi)
    out[..., 0:2, :] = np.einsum("sr,rtzyxic->stzyxic", up, psi[..., 0:2, :])
    out[..., 2:4, :] = np.einsum("sr,rtzyxic->stzyxic", dn, psi[..., 2:4, :])
    return out


def L_op(mob, psi):
    """(L psi)_s = P- psi_{s+1} + P+ psi_{s-1} with the -mf wraps (R1), written out slice by slice."""
    Ls = mob.Ls
    out = np.zeros_like(psi)
    for s in range(Ls):
        up = psi[s - 1] if s >= 1 else -mob.mf * psi[Ls - 1]
        dn = psi[s + 1] if s + 1 < Ls else -mob.mf * psi[0]
        out[s, ..., 0:2, :] = up[..., 0:2, :]   # P+ part
        out[s, ..., 2:4, :] = dn[..., 2:4, :]   # P- part
    return out


def M5(mob, psi, dagger=False):
    return apply_5d(mob.m5_plus(), psi, dagger)


def Mphi(mob, psi, dagger=False):
    return apply_5d(mob.mphi_plus(), psi, dagger)


def M5inv(mob, psi, dagger=False):
    """"a dense matrix multiplication in the fifth dimension" with the closed form R4."""
    return apply_5d(mob.m5inv_plus_closed_form(), psi, dagger)


# ---------------------------------------------------------------------------
# PAPER.md:91 eq. (4) -- the unpreconditioned operator on the full lattice:
#   [[M5, M4eo],[M4oe, M5]]  with  M4 = D^w Mphi  (eq. 7; Mphi first, then the hop)
# ---------------------------------------------------------------------------
def D_dw(mob, U, psi, periodic=(True,) * 4):
    return M5(mob, psi) + hop(U, Mphi(mob, psi), periodic=periodic)


def D_dw_textbook(mob, U, psi):
    """R1 written the other way round: D_DW = (b D_W + 1) + (c D_W - 1) L, D_W = (4-M5) - D^w/2."""
    def D_W(v):
        return (4.0 - mob.M5) * v - 0.5 * hop(U, v)
    Lpsi = L_op(mob, psi)
    return mob.b * D_W(psi) + psi + mob.c * D_W(Lpsi) - Lpsi


# ---------------------------------------------------------------------------
# PAPER.md:95 eq. (5):  D = 1 - M5^-1 M4eo M5^-1 M4oe  on even sites, applied factor by factor.
# PAPER.md:232 eq. (15) (the clean form of the garbled eq. 10, R6): D^dag D as 12 factors.
# The input must be supported on even sites; each hop flips parity, so no masks are needed.
# ---------------------------------------------------------------------------
def D_eo(mob, U, psi_e, periodic=(True,) * 4):
    v = Mphi(mob, psi_e)                     # M_phi
    v = hop(U, v, periodic=periodic)         # D^w        (M4oe = D^w M_phi: even -> odd)
    v = M5inv(mob, v)                        # M5^-1
    v = Mphi(mob, v)                         # M_phi
    v = hop(U, v, periodic=periodic)         # D^w        (M4eo: odd -> even)
    v = M5inv(mob, v)                        # M5^-1
    return psi_e - v


def D_eo_dag(mob, U, psi_e, periodic=(True,) * 4):
    v = M5inv(mob, psi_e, dagger=True)                 # M5^-dag
    v = hop(U, v, dagger=True, periodic=periodic)      # D^w^dag
    v = Mphi(mob, v, dagger=True)                      # M_phi^dag
    v = M5inv(mob, v, dagger=True)                     # M5^-dag
    v = hop(U, v, dagger=True, periodic=periodic)      # D^w^dag
    v = Mphi(mob, v, dagger=True)                      # M_phi^dag
    return psi_e - v


def MdagM(mob, U, psi_e, periodic=(True,) * 4):
    return D_eo_dag(mob, U, D_eo(mob, U, psi_e, periodic), periodic)


# ---------------------------------------------------------------------------
# Full 4-step solve.  PAPER.md:89-97: the 2x2 system of eq. (4),
#   [[M5, M4eo], [M4oe, M5]] (psi_e, psi_o) = (phi_e, phi_o),
# is solved through eq. (5) D psi_e = phihat_e with the prepared source of eq. (6),
#   phihat_e = M5^-1 phi_e - M5^-1 M4eo M5^-1 phi_o,
# the normal equations of eq. (9), D^dag D psi_e = D^dag phihat_e, and the second row of
# eq. (4) for the odd sites, psi_o = M5^-1 (phi_o - M4oe psi_e).  M4 = D^w Mphi (eq. 7).
# Fields carry both parities (the unused one zero), so phi = phi_e + phi_o needs no index code.
# ---------------------------------------------------------------------------
def M4(mob, U, psi):
    """M4eo / M4oe of eq. (7): the hop flips the parity of whatever it is given."""
    return hop(U, Mphi(mob, psi))


def prepare_source(mob, U, phi_e, phi_o):
    """eq. (6): phihat_e."""
    return M5inv(mob, phi_e) - M5inv(mob, M4(mob, U, M5inv(mob, phi_o)))


def normal_rhs(mob, U, phi_e, phi_o):
    """eq. (9): right-hand side D^dag phihat_e of the CGNR system."""
    return D_eo_dag(mob, U, prepare_source(mob, U, phi_e, phi_o))


def reconstruct_odd(mob, U, psi_e, phi_o):
    """Second row of eq. (4): psi_o = M5^-1 (phi_o - M4oe psi_e)."""
    return M5inv(mob, phi_o - M4(mob, U, psi_e))


# ---------------------------------------------------------------------------
# Dirichlet block operator A_s with snake terms.
# PAD (binding reading R10): "the vector is padded in both directions of each
# partitioned dimension by size of two ... the pad region is initialized to zero.  The operators
# in (10) ... are then applied to the padded vector sequentially with zero Dirichlet boundary
# condition on the padded boundary."  Pad sites read links by global periodic index.
# ---------------------------------------------------------------------------
PAD = 2


def block_origins(dims, block):
    Lx, Ly, Lz, Lt = dims
    Bx, By, Bz, Bt = block
    return [(ox, oy, oz, ot)
            for ot in range(0, Lt, Bt) for oz in range(0, Lz, Bz)
            for oy in range(0, Ly, By) for ox in range(0, Lx, Bx)]


def _box_ranges(dims, block, origin):
    """Per direction: (global index array of the padded box, is_cut)."""
    out = []
    for L, B, o in zip(dims, block, origin):
        cut = B != L
        if cut:
            out.append((np.arange(o - PAD, o + B + PAD) % L, True))
        else:
            out.append((np.arange(L), False))
    return out


def box_links(U, dims, block, origin):
    rx, ry, rz, rt = _box_ranges(dims, block, origin)
    Ub = U[:, rt[0]][:, :, rz[0]][:, :, :, ry[0]][:, :, :, :, rx[0]]
    periodic = tuple(not r[1] for r in (rx, ry, rz, rt))
    return Ub, periodic


def box_embed(v_full, dims, block, origin):
    """Copy the block's part of a full-lattice field into the centre of a zero padded box."""
    rx, ry, rz, rt = _box_ranges(dims, block, origin)
    sub = v_full[:, rt[0]][:, :, rz[0]][:, :, :, ry[0]][:, :, :, :, rx[0]].copy()
    for ax, r in zip((4, 3, 2, 1), (rx, ry, rz, rt)):
        if r[1]:
            sl = [slice(None)] * sub.ndim
            sl[ax] = slice(0, PAD)
            sub[tuple(sl)] = 0.0
            sl[ax] = slice(-PAD, None)
            sub[tuple(sl)] = 0.0
    return sub


def box_centre_mask(dims, block):
    shape = []
    sls = []
    for L, B in zip(dims, block):
        if B != L:
            shape.append(B + 2 * PAD)
            sls.append(slice(PAD, PAD + B))
        else:
            shape.append(L)
            sls.append(slice(None))
    m = np.zeros(shape[::-1], dtype=bool)  # [t,z,y,x]
    m[sls[3], sls[2], sls[1], sls[0]] = True
    return m


def box_extract_add(dst_full, box, dims, block, origin):
    """Write the centre of `box` back into the block's sites of the full-lattice field dst_full."""
    Bx, By, Bz, Bt = block
    ox, oy, oz, ot = origin
    sl = []
    for L, B in zip(dims, block):
        sl.append(slice(PAD, PAD + B) if B != L else slice(None))
    c = box[:, sl[3], sl[2], sl[1], sl[0]]
    dst_full[:, ot:ot + Bt, oz:oz + Bz, oy:oy + By, ox:ox + Bx] = c


def A_block_pad(mob, Ubox, periodic, v_box, centre):
    """A_s v for one block in its padded box: the 12 factors of eq. 15, Dirichlet at the box edge, read the centre."""
    w = MdagM(mob, Ubox, v_box, periodic)
    w[:, ~centre] = 0.0
    return w


def A_block_ps(mob, U, dims, block, origin, v_full):
    """(PS) PAPER.md:171 eq. 14: principal sub-matrix R_s (D^dag D) R_s^T of the GLOBAL operator."""
    m = np.zeros(v_full.shape[1:5], dtype=bool)
    Bx, By, Bz, Bt = block
    ox, oy, oz, ot = origin
    m[ot:ot + Bt, oz:oz + Bz, oy:oy + By, ox:ox + Bx] = True
    vin = v_full.copy()
    vin[:, ~m] = 0.0
    w = MdagM(mob, U, vin)
    w[:, ~m] = 0.0
    return w


def A_block_hopwise_truncated(mob, U, dims, block, origin, v_full):
    """NEGATIVE CONTROL (eq. 11 left side, R12): Dirichlet enforced hop by hop -- drops the snake terms."""
    m = np.zeros(v_full.shape[1:5], dtype=bool)
    Bx, By, Bz, Bt = block
    ox, oy, oz, ot = origin
    m[ot:ot + Bt, oz:oz + Bz, oy:oy + By, ox:ox + Bx] = True

    def cut(a):
        a = a.copy()
        a[:, ~m] = 0.0
        return a

    p = cut(v_full)
    v = cut(hop(U, Mphi(mob, p)))
    v = Mphi(mob, M5inv(mob, v))
    v = cut(hop(U, v))
    y = p - M5inv(mob, v)
    v = M5inv(mob, y, dagger=True)
    v = cut(hop(U, v, dagger=True))
    v = M5inv(mob, Mphi(mob, v, dagger=True), dagger=True)
    v = cut(hop(U, v, dagger=True))
    return y - Mphi(mob, v, dagger=True)
