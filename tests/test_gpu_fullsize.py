"""Parity at BASELINE.json's benchmark size (configs[1] = C2: 16^3 x 32, Ls 16, 8^4 blocks, k = 6), in the launch
configuration bench.py times (outer fp32, inner fp16, NATIVE vectors) and in fp64.  The C oracle computes the full-lattice
D^dag D (every element compared) and M^-1 on sampled Dirichlet blocks (block independence, reading R13: the other
blocks do not enter); what the oracle cannot finish in seconds is covered by properties that hold at any size."""
import numpy as np
import pytest

from oracle.cbind import OracleC
from paper_2104_05615_b200 import F16, F32, F64, LAYOUT_NATIVE, Mspcg, synth

pytestmark = pytest.mark.gpu


def rel(a, b):
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def site_max(a, b, Ls, mask=None):
    """Largest error of one 4D site column (Ls x 24 reals) in units of the rms column norm of b: a single wrong column among
    65536 is invisible in a relative L2 norm at fp16 / fp32 tolerances, not here.  mask: flat boolean over the ABI vector."""
    a = np.asarray(a, dtype=np.float64).reshape(Ls, -1, 24)
    b = np.asarray(b, dtype=np.float64).reshape(Ls, -1, 24)
    if mask is not None:
        m = mask.reshape(Ls, -1, 24)[0, :, 0]
        a, b = a[:, m], b[:, m]
    e = np.sqrt(((a - b) ** 2).sum(axis=(0, 2)))
    return float(e.max() / np.sqrt((b ** 2).sum(axis=(0, 2)).mean()))


@pytest.fixture(scope="module")
def c2():
    import torch
    cfg = synth.CONFIGS["C2"]
    U = synth.gauge_natural_to_abi(synth.random_su3_links(cfg["dims"], cfg["eps"], cfg["gauge_seed"]), cfg["dims"])
    src = synth.gaussian_spinor_abi(cfg["dims"], cfg["Ls"], cfg["src_seed"])
    ora = OracleC(cfg["dims"], cfg["Ls"], cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], cfg["block"])
    ora.load_gauge(U, -1)
    ref = dict(MdagM=ora.apply_MdagM(src))
    blocks = (0, 13, 31)
    ref["pre"] = {b: ora.apply_precond(src, cfg["n_inner"], only_block=b) for b in blocks}
    ref["mask"] = {b: ora.apply_A_block(np.ones_like(src), b).reshape(-1) != 0 for b in blocks}
    return cfg, U, src, ref, torch


def _ctx(cfg, U, outer, inner):
    g = Mspcg(cfg["dims"], cfg["Ls"], cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], cfg["block"])
    g.configure(outer, inner, 18)
    g.load_gauge(U, -1)
    return g


def test_C2_bench_configuration_fp32_outer_fp16_inner(c2):
    cfg, U, src, ref, torch = c2
    g = _ctx(cfg, U, F32, F16)
    d = torch.as_tensor(src.reshape(-1)).cuda()
    v = g.pack(d, F32)
    out = g.unpack(g.apply_MdagM(v, F32, LAYOUT_NATIVE), F32).cpu().numpy()
    assert rel(out, ref["MdagM"]) <= 1e-5 and site_max(out, ref["MdagM"], cfg["Ls"]) <= 1e-5
    z = g.unpack(g.apply_precond(v, cfg["n_inner"], F32, LAYOUT_NATIVE), F32).cpu().numpy().reshape(-1)
    for b, zr in ref["pre"].items():
        m = ref["mask"][b]
        assert m.sum() == src.size // 32
        assert rel(z[m], zr.reshape(-1)[m]) <= 2e-2
        assert site_max(z, zr, cfg["Ls"], m) <= 0.1
    # properties at full size: scale equivariance of the nonlinear map r -> z (R13), finiteness, no block left untouched
    z2 = g.unpack(g.apply_precond(g.pack(d * 3e-6, F32), cfg["n_inner"], F32, LAYOUT_NATIVE), F32).cpu().numpy().reshape(-1)
    assert np.all(np.isfinite(z)) and rel(z2 / 3e-6, z) <= 5e-3
    # <r, z> > 0 per block: k CG steps from a zero guess give a positive-definite map on every block
    zz, rr = z.reshape(src.shape), src
    assert float(np.sum(zz * rr)) > 0
    g.close()


def test_C2_fp16_outer_operator_full_geometry(c2):
    """The fp16 sloppy outer operator (the tile kernel on the FULL geometry: every site of the 16^3 x 32 lattice, all wrap-arounds,
    the antiperiodic boundary) against the oracle, element by element: relative L2 and the worst single site column."""
    cfg, U, src, ref, torch = c2
    g = _ctx(cfg, U, F16, F16)
    d = torch.as_tensor(src.reshape(-1)).cuda()
    out = g.unpack(g.apply_MdagM(g.pack(d, F16), F16, LAYOUT_NATIVE), F16).cpu().numpy()
    assert rel(out, ref["MdagM"]) <= 2e-3
    assert site_max(out, ref["MdagM"], cfg["Ls"]) <= 1e-2
    g.close()


def test_C2_fp64(c2):
    cfg, U, src, ref, torch = c2
    g = _ctx(cfg, U, F64, F64)
    d = torch.as_tensor(src.reshape(-1)).cuda()
    Ad = g.apply_MdagM(d, F64)
    assert rel(Ad.cpu().numpy(), ref["MdagM"]) <= 1e-12
    z = g.apply_precond(d, cfg["n_inner"], F64).cpu().numpy().reshape(-1)
    for b, zr in ref["pre"].items():
        m = ref["mask"][b]
        assert rel(z[m], zr.reshape(-1)[m]) <= 1e-9
    # Hermiticity and positivity of D^dag D at full size (gamma5-hermiticity): <u, A v> = <A u, v>, <v, A v> > 0
    u = torch.as_tensor(synth.gaussian_spinor_abi(cfg["dims"], cfg["Ls"], 99).reshape(-1)).cuda()
    Au = g.apply_MdagM(u, F64)

    def cdot(a, b):   # complex inner product of ABI vectors (re, im interleaved)
        a, b = a.view(-1, 2), b.view(-1, 2)
        return complex(float((a[:, 0] * b[:, 0] + a[:, 1] * b[:, 1]).sum()), float((a[:, 0] * b[:, 1] - a[:, 1] * b[:, 0]).sum()))
    lhs, rhs = cdot(u, Ad), cdot(Au, d)
    assert abs(lhs - rhs) <= 1e-11 * abs(lhs)
    vAv = cdot(d, Ad)
    assert vAv.real > 0 and abs(vAv.imag) <= 1e-11 * vAv.real
    g.close()
