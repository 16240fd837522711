"""ORACLE (test infrastructure; the product never imports this): the 8-/16-bit fixed-point storage format of PAPER.md:268-285,
eq. 17, written out step by step.

    "the floating point numbers are stored as 8-bit and 16-bit signed integers, together with a single-precision floating
     point number as the scale for every color-spinor (color(3) x spinor(4) x complex(2) = 24 real numbers):
         floating point = integer / integer-limit x scale                                                        (17)
     In the kernels these fixed-point numbers are unpacked into single precision floating point numbers."

Reading R21 (the paper fixes neither of the three):
  * integer-limit = 2^(bits-1) - 1 (127, 32767): the symmetric range, so that -x and x store as -q and q;
  * scale = the largest |real| of the 24 numbers of the colour-spinor, held in fp32 (a colour-spinor of zeros stores scale 0
    and integers 0);
  * integer = round-half-to-even(x / scale * integer-limit), computed in fp32 (what a cvt.rni of an fp32 product does).

Pins (tests/test_oracle_fixedpoint.py), none of which re-types the formula: the round-trip bound
|x - dq(q(x))| <= scale / (2 limit) (+ fp32 rounding), the element of largest magnitude exact to fp32 rounding, idempotence
dq(q(dq(q(x)))) = dq(q(x)), equivariance under powers of two and under sign, zeros, and a hand-computed example.
"""
import numpy as np


def int_limit(bits):
    if bits not in (8, 16):
        raise ValueError("eq. 17 names 8-bit and 16-bit integers")
    return (1 << (bits - 1)) - 1


def _reals(x):
    """complex [..., 4, 3] -> fp32 reals [..., 24] (spin, colour, re/im)."""
    x = np.asarray(x)
    if x.shape[-2:] != (4, 3):
        raise ValueError("a colour-spinor is the trailing [4 spin, 3 colour] of the field")
    r = np.stack([x.real, x.imag], axis=-1)
    return r.reshape(x.shape[:-2] + (24,)).astype(np.float32)


def quantise(x, bits):
    """eq. 17 read right to left.  x: complex [..., 4, 3].  Returns (integers [..., 24] as int8 / int16, scale [...] fp32)."""
    lim = np.float32(int_limit(bits))
    r = _reals(x)
    scale = np.abs(r).max(axis=-1).astype(np.float32)
    safe = np.where(scale > 0, scale, np.float32(1)).astype(np.float32)
    q = np.rint((r / safe[..., None]).astype(np.float32) * lim)          # np.rint: round half to even
    q = np.where(scale[..., None] > 0, q, 0)
    return q.astype(np.int8 if bits == 8 else np.int16), scale


def dequantise(q, scale, bits):
    """eq. 17 as printed, in fp32: integer / integer-limit x scale.  Returns complex128 [..., 4, 3] holding fp32 values."""
    lim = np.float32(int_limit(bits))
    r = (q.astype(np.float32) / lim).astype(np.float32) * np.asarray(scale, dtype=np.float32)[..., None]
    r = r.astype(np.float32).reshape(q.shape[:-1] + (4, 3, 2)).astype(np.float64)
    return r[..., 0] + 1j * r[..., 1]


def store(x, bits):
    """What a vector holds after being written to and read back from fixed-point storage."""
    q, s = quantise(x, bits)
    return dequantise(q, s, bits)


def cg_fixed_stored(apply_A, r_in, k, bits):
    """k CG steps from a zero guess (eq. 13) with EVERY vector that a step writes -- A p, x, r, p -- passed
    through the fixed-point store ("the matrix multiplication and BLAS operations use the 8-bit and 16-bit
    fixed-point formats"); scalars in fp64.  apply_A maps and returns complex [..., 4, 3] fields."""
    x = np.zeros_like(r_in)
    r = store(r_in, bits)
    p = r.copy()
    rho = np.vdot(r, r).real
    napply = 0
    for _ in range(k):
        if rho == 0.0:
            break
        q = store(apply_A(p), bits)
        napply += 1
        pq = np.vdot(p, q).real
        if not pq > 0.0:
            break
        a = rho / pq
        x = store(x + a * p, bits)
        r = store(r - a * q, bits)
        rho_new = np.vdot(r, r).real
        p = store(r + (rho_new / rho) * p, bits)
        rho = rho_new
    return x, napply


def precond_fixed(pre, r_full, k, bits, blocks=None):
    """z = M^-1 r (eq. 12-14, PAD reading R10) with the vectors of every block's k-step CG in fixed-point storage
    (cg_fixed_stored above).  `pre` is a solvers.BlockPrecond (variant PAD): its padded boxes and block operator are used as they are."""
    from . import mdwf
    if pre.variant != "PAD":
        raise ValueError("precond_fixed follows the PAD reading (R10)")
    z = np.zeros_like(r_full)
    todo = pre.origins if blocks is None else [pre.origins[i] for i in blocks]
    for o in todo:
        Ub, per = pre._box(o)
        rb = mdwf.box_embed(r_full, pre.dims, pre.block, o)
        xb, n = cg_fixed_stored(lambda p: mdwf.A_block_pad(pre.mob, Ub, per, p, pre.centre), rb, k, bits)
        mdwf.box_extract_add(z, xb, pre.dims, pre.block, o)
        pre.napply += n
    return z
