"""Pins for oracle/fixedpoint.py (eq. 17, reading R21).  CPU only.  None of them re-types the formula:
they are properties any correct reading of eq. 17 has, plus one example worked by hand."""
import numpy as np
import pytest

from oracle import fixedpoint as fx
from oracle import mdwf, solvers
from paper_2104_05615_b200 import synth

EPS32 = 2.0 ** -24


def field(shape, seed, spread=0.0):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal(shape + (4, 3)) + 1j * rng.standard_normal(shape + (4, 3))
    if spread:
        x = x * np.exp(spread * rng.standard_normal(shape))[..., None, None]     # colour-spinors of very different size
    return x


def reals(x):
    return np.stack([x.real, x.imag], axis=-1).reshape(x.shape[:-2] + (24,))


@pytest.mark.parametrize("bits", [8, 16])
def test_round_trip_bound_and_exact_maximum(bits):
    lim = fx.int_limit(bits)
    assert lim == {8: 127, 16: 32767}[bits]
    x = field((5, 7), 1, spread=6.0)
    q, s = fx.quantise(x, bits)
    assert q.dtype == (np.int8 if bits == 8 else np.int16) and s.dtype == np.float32 and q.shape == (5, 7, 24)
    assert np.abs(q.astype(np.int64)).max() == lim and np.abs(q.astype(np.int64)).max(axis=-1).min() == lim
    r, d = reals(x), reals(fx.store(x, bits))
    smax = np.abs(r).max(axis=-1)
    assert np.all(np.abs(s - smax) <= 2 * EPS32 * smax)
    # half a step of the grid scale/limit, plus fp32 rounding of the three fp32 operations
    bound = smax[..., None] * (0.5 / lim + 8 * EPS32)
    assert np.all(np.abs(r - d) <= bound)
    # the bound is attained to within a factor 2 somewhere (a format with twice the resolution would not be eq. 17's)
    assert (np.abs(r - d) / smax[..., None]).max() >= 0.25 / lim
    # the largest element of every colour-spinor comes back exactly (to fp32 rounding)
    i = np.abs(r).argmax(axis=-1)[..., None]
    big, bigd = np.take_along_axis(r, i, -1), np.take_along_axis(d, i, -1)
    assert np.all(np.abs(big - bigd) <= 4 * EPS32 * np.abs(big))


@pytest.mark.parametrize("bits", [8, 16])
def test_idempotence_sign_and_power_of_two_equivariance_zeros(bits):
    x = field((11,), 2, spread=3.0)
    once = fx.store(x, bits)
    q1, s1 = fx.quantise(x, bits)
    q2, s2 = fx.quantise(once, bits)
    assert np.array_equal(q1, q2) and np.array_equal(s1, s2)        # stored values are fixed points of the store
    assert np.array_equal(fx.store(once, bits), once)
    qm, sm = fx.quantise(-x, bits)
    assert np.array_equal(qm, -q1) and np.array_equal(sm, s1)       # symmetric integer range
    for e in (-20, 3, 40):
        qe, se = fx.quantise(np.ldexp(1.0, e) * x, bits)
        assert np.array_equal(qe, q1) and np.array_equal(se, np.ldexp(s1, e))
    qc, sc = fx.quantise(np.conj(x), bits)                         # re and im are stored separately
    assert np.array_equal(qc.reshape(-1, 12, 2)[..., 0], q1.reshape(-1, 12, 2)[..., 0])
    assert np.array_equal(qc.reshape(-1, 12, 2)[..., 1], -q1.reshape(-1, 12, 2)[..., 1])
    z = np.zeros((3, 4, 3), dtype=np.complex128)
    qz, sz = fx.quantise(z, bits)
    assert not qz.any() and not sz.any() and not fx.store(z, bits).any()
    # one scale PER colour-spinor: a tiny colour-spinor next to a huge one keeps its relative precision
    y = field((2,), 3)
    y[0] *= 1e-12
    y[1] *= 1e+12
    d = fx.store(y, bits)
    for j in range(2):
        assert np.abs(reals(d[j]) - reals(y[j])).max() <= np.abs(reals(y[j])).max() * (0.5 / fx.int_limit(bits) + 8 * EPS32)


def test_hand_worked_example():
    """A colour-spinor whose largest real is 2: scale = 2, grid step 2/127 (8 bits).
       1.0 -> 1/2*127 = 63.5 -> 64 (half to even) -> 64/127*2 = 1.00787...;  -0.5 -> -31.75 -> -32;  0.01 -> 0.635 -> 1;
       0.0078 -> 0.4953 -> 0;  2 -> 127;  -2 -> -127;  1.5 -> 95.25 -> 95;  0.0236... = 1.5 steps -> 1.5 -> 2 (half to even)."""
    v = np.zeros(24)
    v[:7] = [2.0, -2.0, 1.0, -0.5, 0.01, 0.0078, 1.5]
    v[7] = 1.5 * 2.0 / 127.0
    x = (v[0::2] + 1j * v[1::2]).reshape(4, 3)
    q, s = fx.quantise(x, 8)
    assert s == np.float32(2.0)
    assert list(q[:8]) == [127, -127, 64, -32, 1, 0, 95, 2] and not q[8:].any()
    d = reals(fx.dequantise(q, s, 8))
    assert np.allclose(d[:8], np.array([127, -127, 64, -32, 1, 0, 95, 2]) * 2.0 / 127.0, rtol=1e-6, atol=0)
    q16, s16 = fx.quantise(x, 16)
    assert list(q16[:4]) == [32767, -32767, 16384, -8192] and s16 == np.float32(2.0)     # 16383.5 -> 16384, -8191.75 -> -8192
    with pytest.raises(ValueError):
        fx.int_limit(12)


def test_block_cg_with_stored_vectors_16_bits_close_8_bits_visibly_worse():
    """"Preconditioning kernels with 8-bit fixed-point format ... noticeable impact on the quality of the
    preconditioner ... compared to the 16-bit case".  On a small lattice k CG steps with every vector passed through the store
    stay within 1e-3 of the exact-arithmetic steps at 16 bits and are at least ten times further off at 8 bits."""
    dims, Ls = (4, 4, 4, 4), 4
    mob = mdwf.Mobius(Ls, 1.5, 0.5, 1.8, 0.05)
    U = mdwf.fold_t_boundary(synth.random_su3_links(dims, 0.3, 5), -1)
    r = mdwf.unpack_spinor_abi(synth.gaussian_spinor_abi(dims, Ls, 6), dims, Ls, 0)
    A = lambda v: mdwf.MdagM(mob, U, v)
    ref, n = solvers.cg_fixed(A, r, 5)
    x16, n16 = fx.cg_fixed_stored(A, r, 5, 16)
    x8, n8 = fx.cg_fixed_stored(A, r, 5, 8)
    assert n == n16 == n8 == 5
    e16 = np.linalg.norm(x16 - ref) / np.linalg.norm(ref)
    e8 = np.linalg.norm(x8 - ref) / np.linalg.norm(ref)
    assert e16 <= 1e-3, e16
    assert 10 * e16 <= e8 <= 0.2, (e16, e8)
    # odd sites stay empty through the store (a zero colour-spinor stores as zero)
    assert not mdwf.unpack_spinor_abi(mdwf.pack_spinor_abi(x16, dims, 1), dims, Ls, 1).any()


def test_block_preconditioner_with_stored_vectors():
    """precond_fixed = the PAD block preconditioner with cg_fixed_stored in every block: block independence (R13) survives the store,
    16 bits stays within 1e-3 of the exact-arithmetic preconditioner, 8 bits is at least ten times further off."""
    from oracle import Oracle
    dims, Ls, block, k = (4, 4, 4, 4), 4, (2, 4, 2, 2), 3
    ora = Oracle(dims, Ls, 1.5, 0.5, 1.8, 0.05, block)
    ora.load_gauge(synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.3, 5), dims), -1)
    pre = ora.precond_obj("PAD")
    r = ora.unpack(synth.gaussian_spinor_abi(dims, Ls, 4))
    exact = pre(r, k)
    z16 = fx.precond_fixed(pre, r, k, 16)
    z8 = fx.precond_fixed(pre, r, k, 8)
    e16 = np.linalg.norm(z16 - exact) / np.linalg.norm(exact)
    e8 = np.linalg.norm(z8 - exact) / np.linalg.norm(exact)
    assert 0 < e16 <= 1e-3 and 10 * e16 <= e8 <= 0.2, (e16, e8)
    one = fx.precond_fixed(pre, r, k, 16, blocks=[3])
    sl = np.abs(one).sum(axis=(0, 5, 6)) > 0
    assert sl.any() and np.array_equal(one[:, sl], z16[:, sl])          # a block's result does not depend on the other blocks
    with pytest.raises(ValueError):
        fx.precond_fixed(ora.precond_obj("PS"), r, k, 16)
