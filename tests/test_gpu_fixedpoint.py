"""SURVEY 8(f) f1, eq. 17: the fixed-point storage format on the GPU against oracle/fixedpoint.py.

  * mspcg_fixed_pack / _unpack: integers and scales BIT-IDENTICAL to the oracle's (the rounding decision is taken in fp32 on both sides, R21),
    on a vector whose colour-spinors span 12 orders of magnitude, with zeros and exact ties;
  * mspcg_set_fixed_storage: the fp32-storage preconditioner with r, p, q = A p, x passed through the store inside the kernels, against the
    oracle's block CG with stored vectors (precond_fixed).  The operator runs in fp32 on the GPU and in fp64 in the oracle, so a few
    integers of the stored vectors differ by one unit: tolerance 2e-4 (16 bits: one unit is 3e-5 of the colour-spinor's maximum) and 5e-3
    (8 bits: one unit is 8e-3, fewer flips) in relative L2 -- and both are far from the plain fp32 preconditioner (1e-3 / 5e-2), so the mode
    is really on; 8 bits is visibly worse than 16."""
import numpy as np
import pytest

from oracle import Oracle
from oracle import fixedpoint as fx
from paper_2104_05615_b200 import F32, Mspcg, synth

pytestmark = pytest.mark.gpu

MOB = dict(b=1.5, c=0.5, M5=1.8)


def rel(a, b):
    a, b = np.asarray(a, dtype=np.float64).reshape(-1), np.asarray(b, dtype=np.float64).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.mark.parametrize("bits", [8, 16])
def test_fixed_pack_unpack_bit_identical_to_oracle(bits):
    import torch
    dims, Ls = (4, 4, 6, 2), 6
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.01, dims)
    v = synth.gaussian_spinor_abi(dims, Ls, 7).reshape(-1, 24)
    rng = np.random.default_rng(3)
    v *= np.exp(5.0 * rng.standard_normal(v.shape[0]))[:, None]      # colour-spinors of very different size
    v[5] = 0.0                                                        # an all-zero colour-spinor
    v[6] = 0.0; v[6, 0] = 2.0; v[6, 1] = 1.0; v[6, 2] = -0.5          # exact ties at 8 bits (63.5 -> 64, -31.75 -> -32)
    lim = fx.int_limit(bits)
    v[7] = 0.0; v[7, 0] = 1.0; v[7, 1] = 1.5 / lim; v[7, 2] = 2.5 / lim; v[7, 3] = -0.5 / lim    # ties 1.5 -> 2, 2.5 -> 2, -0.5 -> -0
    d = torch.as_tensor(v.reshape(-1)).cuda()
    q, sc = g.fixed_pack(d, bits)
    # the oracle takes complex [..., 4, 3]; ABI reals are (spin, colour, re/im) in that order
    z = (v[:, 0::2] + 1j * v[:, 1::2]).reshape(-1, 4, 3)
    q_ref, s_ref = fx.quantise(z, bits)
    assert np.array_equal(q.cpu().numpy().reshape(-1, 24), q_ref)
    assert np.array_equal(sc.cpu().numpy(), s_ref)
    back = g.fixed_unpack(q, sc, bits).cpu().numpy().reshape(-1, 24)
    ref = fx.dequantise(q_ref, s_ref, bits)
    ref = np.stack([ref.real, ref.imag], axis=-1).reshape(-1, 24)
    assert np.array_equal(back, ref)
    g.close()


def test_preconditioner_with_fixed_point_vectors_matches_oracle():
    import torch
    dims, Ls, block, k = (4, 4, 4, 8), 8, (4, 4, 2, 4), 4
    U = synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.3, 5), dims)
    ora = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.02, block)
    ora.load_gauge(U, -1)
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.02, block)
    g.configure(F32, F32, 18)
    g.load_gauge(U, -1)
    r = synth.gaussian_spinor_abi(dims, Ls, 9)
    d = torch.as_tensor(r.reshape(-1)).cuda()
    pre = ora.precond_obj("PAD")
    exact = ora.apply_precond(r, k)
    z32 = g.apply_precond(d, k, F32).cpu().numpy()
    assert rel(z32, exact) <= 2e-5                      # plain fp32 storage
    err = {}
    for bits, tol in ((16, 2e-4), (8, 5e-3)):
        ref = ora.pack(fx.precond_fixed(pre, ora.unpack(r), k, bits))
        g.set_fixed_storage(bits)
        z = g.apply_precond(d, k, F32).cpu().numpy()
        assert rel(z, ref) <= tol, (bits, rel(z, ref))
        err[bits] = rel(ref, exact)
        assert rel(z, exact) >= 0.3 * err[bits]          # the store is really applied on the GPU
    g.set_fixed_storage(0)
    assert rel(g.apply_precond(d, k, F32).cpu().numpy(), z32) == 0.0
    assert 1e-5 <= err[16] <= 2e-3 and 10 * err[16] <= err[8] <= 0.3, err
    with pytest.raises(Exception):
        g.set_fixed_storage(12)
    g.close()


def test_fixed_storage_second_geometry_and_scope():
    """Ls 12, a ragged lattice with an uncut direction; and the mode leaves fp16 / fp64 inner storage alone (include/mspcg.h)."""
    import torch
    from paper_2104_05615_b200 import F16, F64
    dims, Ls, block, k = (4, 6, 4, 4), 12, (2, 6, 2, 2), 3
    U = synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.25, 8), dims)
    ora = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.01, block)
    ora.load_gauge(U, -1)
    r = synth.gaussian_spinor_abi(dims, Ls, 10)
    d = torch.as_tensor(r.reshape(-1)).cuda()
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.01, block)
    g.configure(F32, F32, 18)
    g.load_gauge(U, -1)
    g.set_fixed_storage(16)
    ref = ora.pack(fx.precond_fixed(ora.precond_obj("PAD"), ora.unpack(r), k, 16))
    assert rel(g.apply_precond(d, k, F32).cpu().numpy(), ref) <= 2e-4
    g.close()
    for inner in (F16, F64):
        g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.01, block)
        g.configure(F64 if inner == F64 else F32, inner, 18)
        g.load_gauge(U, -1)
        z0 = g.apply_precond(d, k, F64).cpu().numpy()
        g.set_fixed_storage(8)
        # not bitwise: the per-block scalars are summed with atomics; an 8-bit store would show at the 1e-2 level
        assert rel(g.apply_precond(d, k, F64).cpu().numpy(), z0) <= (1e-12 if inner == F64 else 2e-3)
        g.close()
