"""GPU parity tests: the CUDA library (through its C ABI) against the CPU oracle, element by element, same seeded inputs.

Tolerances (BASELINE.json north_star):
  operator apply   rel-L2 <= 1e-12 (fp64), <= 1e-5 (fp32), <= 2e-3 (fp16 storage / fp32 arithmetic)
  M_pre apply      rel-L2 <= 1e-9 (fp64, k <= 8: CG amplifies summation-order differences), 2e-2 (fp16)
  solve            true fp64 residual <= 1e-10, solution within 1e-8 (relative) of the oracle's
"""
import numpy as np
import pytest

from oracle.cbind import OracleC
from paper_2104_05615_b200 import F16, F32, F64, LAYOUT_NATIVE, Mspcg, MspcgError, synth

pytestmark = pytest.mark.gpu

MOB = dict(b=1.5, c=0.5, M5=1.8)


def rel(a, b):
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def setup(dims, Ls, mf, block, eps=0.3, gauge_seed=5, outer=F64, inner=F64, recon=18, tb=-1):
    import torch
    U = synth.gauge_natural_to_abi(synth.random_su3_links(dims, eps, gauge_seed), dims)
    ora = OracleC(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf, block)
    ora.load_gauge(U, tb)
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf, block)
    g.configure(outer, inner, recon)
    g.load_gauge(U, tb)
    return ora, g, torch


def dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64).reshape(-1)).cuda()


# lattice, Ls, block: several thread-block tiles, ragged tails (site counts not multiples of the 8/16/32-site tile),
# an uncut direction, blocks touching the antiperiodic boundary, and the wrap-around case L - B < 4 (PAD != PS, R10).
GEOMS = [
    ((4, 4, 4, 4), 8, (2, 2, 2, 2)),      # C1 geometry
    ((2, 4, 6, 6), 4, (2, 2, 6, 2)),      # ragged, y partially cut, z uncut
    ((8, 4, 4, 6), 6, (4, 4, 2, 6)),      # t uncut
    ((4, 4, 4, 8), 12, (4, 2, 4, 4)),
    ((4, 6, 4, 4), 16, (2, 6, 2, 2)),
]


def test_pack_unpack_roundtrip():
    ora, g, torch = setup((4, 4, 6, 2), 6, 0.01, (2, 2, 2, 2))
    v = synth.gaussian_spinor_abi((4, 4, 6, 2), 6, 3)
    d = dev(torch, v)
    for prec, tol in ((F64, 0.0), (F32, 1e-7), (F16, 1e-3)):
        back = g.unpack(g.pack(d, prec), prec).cpu().numpy()
        assert rel(back, v) <= tol


@pytest.mark.parametrize("dims,Ls,block", GEOMS)
def test_MdagM_fp64(dims, Ls, block):
    ora, g, torch = setup(dims, Ls, 0.02, block)
    v = synth.gaussian_spinor_abi(dims, Ls, 7)
    out = g.apply_MdagM(dev(torch, v), F64).cpu().numpy()
    assert rel(out, ora.apply_MdagM(v)) <= 1e-12


@pytest.mark.parametrize("tb", [+1, -1])
def test_MdagM_fp64_boundary_and_unit_gauge(tb):
    import torch
    dims, Ls = (4, 4, 4, 6), 8
    U = synth.gauge_natural_to_abi(synth.unit_links(dims), dims)
    ora = OracleC(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.05, dims)
    ora.load_gauge(U, tb)
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.05, dims)
    g.configure(F64, F64, 18)
    g.load_gauge(U, tb)
    v = synth.gaussian_spinor_abi(dims, Ls, 8)
    assert rel(g.apply_MdagM(dev(torch, v), F64).cpu().numpy(), ora.apply_MdagM(v)) <= 1e-12


@pytest.mark.parametrize("prec,tol,recon", [(F32, 1e-5, 18), (F16, 2e-3, 18), (F32, 1e-5, 12), (F16, 2e-3, 12)])
def test_MdagM_low_precision(prec, tol, recon):
    dims, Ls, block = (4, 4, 6, 8), 8, (2, 2, 6, 4)
    ora, g, torch = setup(dims, Ls, 0.02, block, outer=prec, inner=prec, recon=recon)
    v = synth.gaussian_spinor_abi(dims, Ls, 9)
    ref = ora.apply_MdagM(v)
    d = dev(torch, v)
    assert rel(g.apply_MdagM(d, prec).cpu().numpy(), ref) <= tol
    nat = g.pack(d, prec)
    out = g.unpack(g.apply_MdagM(nat, prec, LAYOUT_NATIVE), prec).cpu().numpy()
    assert rel(out, ref) <= tol


@pytest.mark.parametrize("dims,Ls,block", [((4, 4, 4, 8), 4, (2, 2, 4, 4)), ((4, 4, 6, 4), 6, (2, 2, 2, 2)),
                                           ((8, 4, 4, 8), 12, (4, 4, 2, 4)), ((4, 8, 4, 8), 16, (4, 4, 4, 4))])
def test_fp16_tensor_core_hop_every_compiled_Ls(dims, Ls, block):
    """The fp16 path (half-spinor projection, SU(3) and Ls x Ls contractions on the tensor cores) at every compiled Ls: one and
    two row segments, partially filled second segment (Ls = 12), full lattice and Dirichlet blocks."""
    ora, g, torch = setup(dims, Ls, 0.02, block, outer=F16, inner=F16)
    v = synth.gaussian_spinor_abi(dims, Ls, 19)
    assert rel(g.apply_MdagM(dev(torch, v), F16).cpu().numpy(), ora.apply_MdagM(v)) <= 2e-3
    assert rel(g.apply_precond(dev(torch, v), 6, F64).cpu().numpy(), ora.apply_precond(v, 6)) <= 2e-2


@pytest.mark.parametrize("dims,Ls,block", GEOMS)
def test_A_block_fp64(dims, Ls, block):
    ora, g, torch = setup(dims, Ls, 0.02, block)
    v = synth.gaussian_spinor_abi(dims, Ls, 11)
    d = dev(torch, v)
    nblk = g.geometry()["nblk"]
    assert nblk == ora.num_blocks
    for blk in sorted({0, nblk // 2, nblk - 1}):
        out = g.apply_A_block(d, blk, F64).cpu().numpy()
        assert rel(out, ora.apply_A_block(v, blk)) <= 1e-12


@pytest.mark.parametrize("dims,Ls,block", GEOMS)
@pytest.mark.parametrize("k", [1, 4])
def test_precond_fp64(dims, Ls, block, k):
    ora, g, torch = setup(dims, Ls, 0.02, block)
    r = synth.gaussian_spinor_abi(dims, Ls, 13)
    z = g.apply_precond(dev(torch, r), k, F64).cpu().numpy()
    assert rel(z, ora.apply_precond(r, k)) <= 1e-9


def test_precond_degenerate_inputs():
    dims, Ls, block = (4, 4, 4, 4), 8, (2, 2, 2, 2)
    ora, g, torch = setup(dims, Ls, 0.02, block)
    r = synth.gaussian_spinor_abi(dims, Ls, 14)
    # zero right-hand side -> zero, never NaN (R13)
    z0 = g.apply_precond(dev(torch, 0 * r), 6, F64).cpu().numpy()
    assert np.all(z0 == 0.0)
    # one block's right-hand side zero: that block returns zero, the others are untouched (block independence)
    rr = r.copy()
    mask = ora.apply_A_block(np.ones_like(r), 5) != 0  # support of block 5
    rr[mask] = 0.0
    z = g.apply_precond(dev(torch, rr), 4, F64).cpu().numpy().reshape(r.shape)
    zr = ora.apply_precond(rr, 4).reshape(r.shape)
    assert np.all(z[mask] == 0.0) and rel(z, zr) <= 1e-9
    # scale equivariance z(lambda r) = lambda z(r)
    z1 = g.apply_precond(dev(torch, r), 3, F64).cpu().numpy()
    z2 = g.apply_precond(dev(torch, 1e-7 * r), 3, F64).cpu().numpy()
    assert rel(z2 * 1e7, z1) <= 1e-10
    # k >> dimension of the Krylov space that matters: many iterations stay finite
    zk = g.apply_precond(dev(torch, r), 32, F64).cpu().numpy()
    assert np.all(np.isfinite(zk))


@pytest.mark.parametrize("inner,tol", [(F32, 2e-4), (F16, 2e-2)])
def test_precond_low_precision(inner, tol):
    dims, Ls, block = (4, 4, 8, 8), 8, (4, 4, 4, 4)
    ora, g, torch = setup(dims, Ls, 0.02, block, outer=F32, inner=inner)
    r = synth.gaussian_spinor_abi(dims, Ls, 15)
    ref = ora.apply_precond(r, 6)
    z = g.apply_precond(dev(torch, r), 6, F64).cpu().numpy()
    assert rel(z, ref) <= tol
    # tiny right-hand side: the per-block rescaling keeps fp16 in range (R14)
    z = g.apply_precond(dev(torch, 1e-9 * r), 6, F64).cpu().numpy()
    assert rel(z * 1e9, ref) <= tol


def test_solve_C1_cg_and_mspcg_fp64():
    """BASELINE.json configs[0]: 4^4, Ls 8, mf 0.01, 2^4 blocks, 6 inner iterations, tol 1e-10."""
    cfg = synth.CONFIGS["C1"]
    dims, Ls, block = cfg["dims"], cfg["Ls"], cfg["block"]
    ora, g, torch = setup(dims, Ls, cfg["mf"], block, eps=cfg["eps"], gauge_seed=cfg["gauge_seed"])
    b = synth.gaussian_spinor_abi(dims, Ls, cfg["src_seed"])
    x_ora, so = ora.solve(b, tol=1e-10, use_precond=False)
    x_orap, sop = ora.solve(b, tol=1e-10, use_precond=True, n_inner=cfg["n_inner"])
    db = dev(torch, b)
    x, s = g.solve(db, tol=1e-10, use_precond=False)
    xp, spc = g.solve(db, tol=1e-10, use_precond=True, n_inner=cfg["n_inner"])
    for xx, ss in ((x, s), (xp, spc)):
        assert ss["rc"] == 0 and ss["converged"] == 1
        assert ss["true_res"] <= 1e-10
        # independent check of the residual with the oracle's operator
        xn = xx.cpu().numpy()
        assert rel(ora.apply_MdagM(xn), b) <= 1e-10 * 1.01
        assert rel(xn, x_ora) <= 1e-8
    assert rel(x_orap, x_ora) <= 1e-8
    # iteration counts against the oracle's (eq. 18 beta on both sides): the library looks at |r| one iteration late (R15b),
    # so it may run one iteration more; rounding order accounts for the other one
    assert abs(s["iters"] - so["iters"]) <= 2, (s["iters"], so["iters"])
    assert abs(spc["iters"] - sop["iters"]) <= 2, (spc["iters"], sop["iters"])
    assert spc["iters"] < s["iters"]
    assert spc["inner_applies"] > 0


def test_solve_mixed_precision_reliable_updates():
    dims, Ls, block = (4, 4, 4, 8), 8, (2, 2, 2, 4)
    ora, g, torch = setup(dims, Ls, 0.01, block, eps=0.3, outer=F32, inner=F16)
    b = synth.gaussian_spinor_abi(dims, Ls, 17)
    x_ora, _ = ora.solve(b, tol=1e-11, use_precond=False)
    db = dev(torch, b)
    for pre in (False, True):
        x, s = g.solve(db, tol=1e-10, use_precond=pre, n_inner=5, sloppy_prec=F32, delta=0.1)
        assert s["rc"] == 0 and s["true_res"] <= 1e-10 and s["reliable_updates"] >= 2
        assert rel(x.cpu().numpy(), x_ora) <= 1e-8
    # zero right-hand side and a non-zero initial guess
    x, s = g.solve(0 * db, tol=1e-10)
    assert s["converged"] == 1 and s["iters"] == 0 and float(x.abs().max()) == 0.0
    x, s = g.solve(db, x0_abi=dev(torch, x_ora), tol=1e-10)
    assert s["converged"] == 1 and s["iters"] <= 1


@pytest.mark.parametrize("inner,tol", [(F64, 1e-12), (F16, 2e-3)])
def test_block_groups_give_the_same_preconditioner(inner, tol):
    """the L2-resident schedule (all inner iterations for G blocks at a time, same buffers for every group) changes
    the order of work only: blocks are independent (R13).  16 blocks in groups of 3 (ragged last group) and of 1, against the
    oracle and against the ungrouped result; the reduced-Ls path too."""
    from oracle import Oracle, reduced_ls
    dims, Ls, block, k = (4, 8, 4, 8), 8, (2, 4, 2, 4), 4
    import torch
    U = synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.3, 5), dims)
    ora = OracleC(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.02, block)
    ora.load_gauge(U, -1)
    T = reduced_ls.initial_T(Ls, 4)
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.02, block)
    g.set_reduced_ls(4, reduced_ls.T_to_abi(T), 0.5)
    g.configure(F64 if inner == F64 else F32, inner, 18)
    g.load_gauge(U, -1)
    r = synth.gaussian_spinor_abi(dims, Ls, 11)
    d = dev(torch, r)
    ref = ora.apply_precond(r, k)
    z0 = g.apply_precond(d, k, F64).cpu().numpy()
    zr0 = g.apply_precond(d, k, F64, use_reduced=1).cpu().numpy()
    assert rel(z0, ref) <= (1e-9 if inner == F64 else 2e-2)
    for G in (3, 1):
        g.set_block_group(G)
        assert rel(g.apply_precond(d, k, F64).cpu().numpy(), z0) <= tol
        assert rel(g.apply_precond(d, k, F64, use_reduced=1).cpu().numpy(), zr0) <= tol
    x, st = g.solve(d, tol=1e-10, use_precond=True, n_inner=k, sloppy_prec=F64 if inner == F64 else F32)
    assert st["rc"] == 0 and st["true_res"] <= 1e-10
    g.close()


@pytest.mark.parametrize("inner", [F64, F16])
def test_poisoned_neighbour_blocks_do_not_leak(inner):
    """Stand-in for the memory checker the GPU pool refuses: every input element OUTSIDE one Dirichlet block is NaN.
    A_s and M^-1 of that block read nothing but the block ("without communication"; the snake terms are temporaries computed
    from the block's own sites), so its output must be finite and what it is with clean neighbours; any read past
    the block -- a wrong neighbour index, a tile slot of another block, a run one column too long -- turns it into NaN."""
    dims, Ls, block, k = (8, 4, 8, 8), 8, (4, 2, 4, 4), 3
    ora, g, torch = setup(dims, Ls, 0.02, block, outer=F64 if inner == F64 else F32, inner=inner)
    v = synth.gaussian_spinor_abi(dims, Ls, 4)
    d = dev(torch, v)
    for blk in (0, 5, ora.num_blocks - 1):
        mask = torch.as_tensor(ora.apply_A_block(np.ones_like(v), blk).reshape(-1) != 0).cuda()   # the block's own sites
        assert int(mask.sum()) == v.size // ora.num_blocks
        poisoned = torch.where(mask, d, torch.full_like(d, float("nan")))
        clean = torch.where(mask, d, torch.zeros_like(d))
        if inner == F64:
            a_p, a_c = g.apply_A_block(poisoned, blk, F64), g.apply_A_block(clean, blk, F64)
            assert bool(torch.isfinite(a_p).all()) and bool((a_p == a_c).all())
        z_p, z_c = g.apply_precond(poisoned, k, F64), g.apply_precond(clean, k, F64)
        assert bool(torch.isfinite(z_p[mask]).all())
        # equal up to the order of the atomic partial sums of the block's inner products
        assert rel(z_p[mask].cpu().numpy(), z_c[mask].cpu().numpy()) <= (1e-12 if inner == F64 else 2e-3)
        assert bool(torch.isnan(z_p[~mask]).any())            # the poison did reach the other blocks' own solves (the test has teeth)
    g.close()


def test_host32_entry_points_match_the_fp64_wire_format():
    """mspcg_apply_*_host32 (float host vectors in the ABI layout) against the fp64 *_host calls and the oracle."""
    dims, Ls, block, k = (4, 4, 6, 8), 8, (2, 2, 6, 4), 3
    ora, g, torch = setup(dims, Ls, 0.02, block, outer=F32, inner=F16)
    v = synth.gaussian_spinor_abi(dims, Ls, 12)
    h64 = torch.as_tensor(v.reshape(-1)).pin_memory()
    h32 = h64.to(torch.float32).pin_memory()
    o64, o32 = torch.empty_like(h64).pin_memory(), torch.empty_like(h32).pin_memory()
    g.apply_MdagM_host(h64, o64, F32)
    g.apply_MdagM_host32(h32, o32, F32)
    assert rel(o32.numpy(), o64.numpy()) <= 2e-7 and rel(o32.numpy(), ora.apply_MdagM(v)) <= 1e-5
    g.apply_precond_host(h64, o64, k, F32)
    g.apply_precond_host32(h32, o32, k, F32)
    assert rel(o32.numpy(), o64.numpy()) <= 2e-3 and rel(o32.numpy(), ora.apply_precond(v, k)) <= 2e-2
    with pytest.raises(MspcgError):
        g.apply_MdagM_host32(h32, o32, F64)
    g.close()


def test_error_codes():
    import torch
    g = Mspcg((4, 4, 4, 4), 8, 1.5, 0.5, 1.8, 0.01, (2, 2, 2, 2))
    v = torch.zeros(g.nreal, dtype=torch.float64, device="cuda")
    from paper_2104_05615_b200 import MspcgError
    with pytest.raises(MspcgError) as e:
        g.apply_MdagM(v, F64)
    assert e.value.code == -7  # no workspace
    g.configure(F64, F64, 18)
    with pytest.raises(MspcgError) as e:
        g.apply_MdagM(v, F64)
    assert e.value.code == -4  # no gauge
    with pytest.raises(MspcgError):
        Mspcg((4, 4, 4, 5), 8, 1.5, 0.5, 1.8, 0.01)
    with pytest.raises(MspcgError):
        Mspcg((4, 4, 4, 4), 8, 1.5, 0.5, 1.8, 0.01, (3, 2, 2, 2))


# ---- reduced-Ls preconditioner (eq. 19-21) against oracle/reduced_ls.py -----------
def _reduced_setup(dims, Ls, Lh, block, mu, inner, outer=F64, seed=21):
    import torch
    from oracle import Oracle, reduced_ls
    U = synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.3, 5), dims)
    hat = Oracle(dims, Lh, MOB["b"], MOB["c"], MOB["M5"], 0.02, block)
    hat.load_gauge(U, -1)
    full = Oracle(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.02, block)
    rng = np.random.default_rng(seed)
    T = reduced_ls.initial_T(Ls, Lh) + 0.2 * (rng.standard_normal((Lh, 4, Ls, 4)) + 1j * rng.standard_normal((Lh, 4, Ls, 4)))
    pre = reduced_ls.ReducedLsPrecond(hat.precond_obj(), T, mu)
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.02, block)
    g.set_reduced_ls(Lh, reduced_ls.T_to_abi(T), mu)
    g.configure(outer, inner, 18)
    g.load_gauge(U, -1)
    return full, pre, g, torch


@pytest.mark.parametrize("dims,Ls,Lh,block", [((4, 4, 4, 4), 8, 4, (2, 2, 4, 4)), ((4, 4, 2, 6), 12, 6, (2, 2, 2, 6)),
                                              ((4, 2, 4, 4), 6, 6, (2, 2, 2, 2))])
def test_reduced_ls_precond_fp64(dims, Ls, Lh, block):
    full, pre, g, torch = _reduced_setup(dims, Ls, Lh, block, 0.4, F64)
    r = synth.gaussian_spinor_abi(dims, Ls, 23)
    ref = full.pack(pre(full.unpack(r), 3))
    z = g.apply_precond(dev(torch, r), 3, F64, use_reduced=1).cpu().numpy()
    assert rel(z, ref) <= 1e-9
    # the full-Ls preconditioner of the same context is untouched by set_reduced_ls
    ora = OracleC(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.02, block)
    ora.load_gauge(synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.3, 5), dims), -1)
    assert rel(g.apply_precond(dev(torch, r), 3, F64).cpu().numpy(), ora.apply_precond(r, 3)) <= 1e-9


def test_reduced_ls_precond_fp16_and_solve():
    dims, Ls, Lh, block = (4, 4, 4, 8), 8, 4, (4, 4, 4, 4)
    full, pre, g, torch = _reduced_setup(dims, Ls, Lh, block, 0.5, F16, outer=F32)
    r = synth.gaussian_spinor_abi(dims, Ls, 25)
    ref = full.pack(pre(full.unpack(r), 4))
    z = g.apply_precond(dev(torch, r), 4, F64, use_reduced=1).cpu().numpy()
    assert rel(z, ref) <= 2e-2
    # MSPCG with the reduced-Ls preconditioner converges to the solution of the same system
    ora = OracleC(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], 0.02, block)
    ora.load_gauge(synth.gauge_natural_to_abi(synth.random_su3_links(dims, 0.3, 5), dims), -1)
    x_ref, _ = ora.solve(r, tol=1e-11)
    x, st = g.solve(dev(torch, r), tol=1e-10, use_precond=True, n_inner=4, sloppy_prec=F32, use_reduced_ls=True)
    assert st["rc"] == 0 and st["true_res"] <= 1e-10 and rel(x.cpu().numpy(), x_ref) <= 1e-8


@pytest.mark.parametrize("dims,Ls,Lh,block", [((4, 4, 4, 8), 8, 4, (4, 4, 4, 4)), ((8, 4, 4, 6), 12, 6, (4, 4, 4, 6)),
                                              ((4, 4, 6, 8), 16, 8, (2, 4, 6, 4))])
def test_reduced_ls_transfer_on_tcgen05_matches_generic_kernels(dims, Ls, Lh, block, monkeypatch):
    """The tcgen05 transfer kernels (fp16 operands, fp32 accumulation in tensor memory) against the generic CUDA-core
    ones (MSPCG_TRANSFER_TC=0) and against the oracle; tile tails: nE0 per block is not a multiple of 128."""
    r = synth.gaussian_spinor_abi(dims, Ls, 27)
    out = {}
    for flag in ("1", "0"):
        monkeypatch.setenv("MSPCG_TRANSFER_TC", flag)
        full, pre, g, torch = _reduced_setup(dims, Ls, Lh, block, 0.3, F16, outer=F32)
        out[flag] = g.apply_precond(dev(torch, r), 4, F64, use_reduced=1).cpu().numpy()
        nat = g.pack(dev(torch, r), F32)
        out[flag + "f32"] = g.unpack(g.apply_precond(nat, 4, F32, LAYOUT_NATIVE, use_reduced=1), F32).cpu().numpy()
        g.close()
    ref = full.pack(pre(full.unpack(r), 4))
    for k in out:
        assert rel(out[k], ref) <= 2e-2
    assert rel(out["1"], out["0"]) <= 5e-3 and rel(out["1f32"], out["0f32"]) <= 5e-3


def test_solve_fp16_sloppy_outer_iteration():
    """fp16 storage of the outer iteration's r, x, p (BASELINE.json configs[4]: "outer fp32/fp16 with fp64 reliable updates"):
    the vectors are rescaled at every residual replacement, so fp16 never underflows on the way to 1e-10."""
    dims, Ls, block = (4, 4, 4, 8), 8, (2, 2, 2, 4)
    ora, g, torch = setup(dims, Ls, 0.01, block, eps=0.3, outer=F16, inner=F16)
    b = synth.gaussian_spinor_abi(dims, Ls, 17)
    x_ora, _ = ora.solve(b, tol=1e-11, use_precond=False)
    for scale in (1.0, 1e-12):     # a tiny right-hand side must not matter
        db = dev(torch, b * scale)
        for pre in (False, True):
            x, s = g.solve(db, tol=1e-10, use_precond=pre, n_inner=5, sloppy_prec=F16, delta=0.1)
            assert s["rc"] == 0 and s["true_res"] <= 1e-10 and s["reliable_updates"] >= 5
            assert rel(x.cpu().numpy() / scale, x_ora) <= 1e-8


def test_precond_fp16_more_blocks_than_resident_thread_blocks():
    """864 Dirichlet blocks > 4 x 148 resident thread blocks: the fp16 hop kernel walks several blocks per thread block."""
    dims, Ls, block = (12, 12, 12, 8), 4, (2, 2, 2, 2)
    ora, g, torch = setup(dims, Ls, 0.02, block, outer=F32, inner=F16)
    assert g.geometry()["nblk"] == 864
    r = synth.gaussian_spinor_abi(dims, Ls, 19)
    z = g.apply_precond(dev(torch, r), 3, F64).cpu().numpy()
    assert rel(z, ora.apply_precond(r, 3)) <= 2e-2


# ---- the dense fifth-dimension contraction on its own: tcgen05 GEMM on an fp16 NATIVE vector ----
@pytest.mark.parametrize("dims,Ls", [((4, 4, 4, 8), 8), ((6, 6, 6, 10), 12), ((8, 8, 6, 6), 16)])
@pytest.mark.parametrize("dagger", [False, True])
def test_M5inv_tcgen05_fp16(dims, Ls, dagger):
    """mspcg_apply_M5inv against the oracle's M5^-1 (closed form R4) applied to the fp16-rounded input.
    Site counts 256, 1080 and 1152: several 128-site tiles and a ragged tail.  Tolerance: the operands and the result are
    rounded to fp16 (2^-11 each), accumulation is fp32 -> 2e-3 as for every fp16-storage operator."""
    import torch
    from oracle import mdwf
    mf = 0.01
    g = Mspcg(dims, Ls, MOB["b"], MOB["c"], MOB["M5"], mf, dims)
    g.configure(F32, F16, 18)
    v = synth.gaussian_spinor_abi(dims, Ls, 11)
    nat = g.pack(dev(torch, v), F16)
    v16 = g.unpack(nat, F16).cpu().numpy()                      # the rounded input, as the kernel sees it
    out = g.unpack(g.apply_M5inv(nat, dagger), F16).cpu().numpy()
    mob = mdwf.Mobius(Ls, MOB["b"], MOB["c"], MOB["M5"], mf)
    ref = mdwf.pack_spinor_abi(mdwf.M5inv(mob, mdwf.unpack_spinor_abi(v16, dims, Ls), dagger), dims)
    assert rel(out, ref) <= 2e-3
    # M5^-1 M5 = 1 (north_star pin) seen from the GPU side: M5 of the oracle on the GPU result gives the input back
    back = mdwf.pack_spinor_abi(mdwf.M5(mob, mdwf.unpack_spinor_abi(out, dims, Ls), dagger), dims)
    assert rel(back, v16) <= 2e-3
    g.close()
