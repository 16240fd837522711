"""Oracle comparisons at the FULL sizes of BASELINE.json configs C3, C4 and C5 (north_star: "on all five configs"), in the
precisions bench.py runs them in.  The oracle cannot apply the whole operator at these sizes in seconds, so it computes
SAMPLED OUTPUTS one by one, which locality makes exact:

  * D^dag D is a product of four nearest-neighbour hops: its output on a 4^4 core of sites depends only on inputs and
    links within 4 hops.  A 12^4 WINDOW of the big lattice (links, boundary sign and source cut out around the core) is
    handed to the oracle as a small periodic lattice; on the core (window coordinates 4..7) the window's own wrap-around
    cannot be felt, so the oracle's output there IS the big-lattice output.
  * M^-1 on one Dirichlet block depends only on the links of the block and its pad of two (reading R10):
    C3 and C4 use the oracle on the full lattice for ONE block (block independence, R13); C5 (too large for the host) rebuilds
    the block and its pad as block 0 of a 2B-periodic lattice, which has identical links on every site the padded box reads.

Every fp16 / fp32 comparison carries a per-site maximum-norm bound next to the relative L2 norm: one wrong site column in
millions is invisible in a global norm at these tolerances.  C5's gauge field is a C2-sized seeded field tiled 3x3x3x3
(generating 42 M independent links takes minutes on the host); the source is not periodic.  Marked slow.
"""
import numpy as np
import pytest

from oracle.cbind import OracleC
from paper_2104_05615_b200 import F16, F32, F64, LAYOUT_NATIVE, Mspcg, synth

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

W = 12   # window extent


def rel(a, b):
    a, b = np.asarray(a, dtype=np.float64).reshape(-1), np.asarray(b, dtype=np.float64).reshape(-1)
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def site_max(a, b):
    """max over 4D sites of |a - b| on the site's Ls x 24 column, in units of the rms column norm of b.  a, b: [Ls, n, 24]."""
    e = np.sqrt(((a - b) ** 2).sum(axis=(0, 2)))
    return float(e.max() / np.sqrt((b ** 2).sum(axis=(0, 2)).mean()))


def window_sites(dims, origin, ext):
    """Global x_cb of the EVEN sites of the box [origin, origin + ext) (periodic), in the ABI order of the box taken as a
    lattice of its own (origin must be even), plus the box-local coordinates."""
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(*(np.arange(e) for e in ext[::-1]), indexing="ij")
    loc = np.stack([x, y, z, t], axis=-1).reshape(-1, 4)
    ev = loc[(loc.sum(axis=1) % 2) == 0]
    g = (ev + np.asarray(origin)) % np.asarray(dims)
    lex = g[:, 0] + Lx * (g[:, 1] + Ly * (g[:, 2] + Lz * g[:, 3]))
    return lex // 2, ev


def cut_links(U, dims, origin, ext, tb=-1):
    """Natural-order links of the box [origin, origin + ext) of the periodic lattice; the antiperiodic sign of the big
    lattice's time boundary is folded into the cut-out links (the small lattice is then run with t_boundary = +1)."""
    idx = [(np.arange(e) + o) % L for e, o, L in zip(ext, origin, dims)]
    sub = U[:, idx[3]][:, :, idx[2]][:, :, :, idx[1]][:, :, :, :, idx[0]].copy()
    if tb == -1:
        sub[3, idx[3] == dims[3] - 1] *= -1.0
    return sub


def window_oracle(cfg, U, origin, ext, block=None):
    ora = OracleC(tuple(ext), cfg["Ls"], cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], tuple(block) if block else tuple(ext))
    ora.load_gauge(synth.gauge_natural_to_abi(cut_links(U, cfg["dims"], origin, ext), tuple(ext)), +1)
    return ora


def check_MdagM_windows(cfg, U, src, out_of, origins, tol, tol_site):
    """out_of(x_cb index array) -> GPU D^dag D output rows [Ls, n, 24] at those even sites."""
    dims, Ls = cfg["dims"], cfg["Ls"]
    for o in origins:
        xcb, loc = window_sites(dims, o, (W,) * 4)
        ora = window_oracle(cfg, U, o, (W,) * 4)
        ref = ora.apply_MdagM(np.ascontiguousarray(src[:, xcb])).reshape(Ls, -1, 24)
        core = np.all((loc >= 4) & (loc <= 7), axis=1)
        got = out_of(xcb[core]).reshape(Ls, -1, 24)
        assert core.sum() == 128
        assert rel(got, ref[:, core]) <= tol, (o, rel(got, ref[:, core]))
        assert site_max(got, ref[:, core]) <= tol_site, (o, site_max(got, ref[:, core]))


def make(cfg, outer, inner, recon=18, U_nat=None):
    import torch
    dims = cfg["dims"]
    U = synth.random_su3_links(dims, cfg["eps"], cfg["gauge_seed"]) if U_nat is None else U_nat
    src = synth.gaussian_spinor_abi(dims, cfg["Ls"], cfg["src_seed"])
    g = Mspcg(dims, cfg["Ls"], cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], cfg["block"])
    g.configure(outer, inner, recon)
    Uabi = synth.gauge_natural_to_abi(U, dims)
    g.load_gauge(Uabi, -1)
    return g, U, Uabi, src, torch


def gpu_rows(torch, v_abi_dev, Ls):
    """Row gather from a device ABI vector: x_cb indices -> numpy [Ls, n, 24]."""
    v = v_abi_dev.view(Ls, -1, 24)
    return lambda xcb: v[:, torch.as_tensor(xcb, device=v.device)].cpu().numpy()


def block_xcb(cfg, blk_origin):
    return window_sites(cfg["dims"], blk_origin, cfg["block"])[0]


@pytest.mark.parametrize("name", ["C3", "C4"])
def test_C3_C4_operator_windows_and_one_block_preconditioner(name):
    """C3 (24^3 x 64, Ls 16, 12^3 x 16 blocks, k 5) and C4 (32^3 x 64, Ls 12, 16^3 x 32 blocks, k 6): sloppy fp32 D^dag D, fp16
    D^dag D on the full lattice and the fp16-storage preconditioner of one block, as bench.py configures them."""
    cfg = synth.CONFIGS[name]
    dims, Ls, block, k = cfg["dims"], cfg["Ls"], cfg["block"], cfg["n_inner"]
    g, U, Uabi, src, torch = make(cfg, F32, F16)
    d = torch.as_tensor(src.reshape(-1)).cuda()
    origins = [(2, 4, 6, 8), (dims[0] - 6, block[1] - 6, 0, dims[3] - 6), (block[0] - 6, block[1] - 6, block[2] - 6, block[3] - 6)]
    out32 = g.unpack(g.apply_MdagM(g.pack(d, F32), F32, LAYOUT_NATIVE), F32)
    check_MdagM_windows(cfg, U, src, gpu_rows(torch, out32, Ls), origins, 1e-5, 1e-5)
    del out32
    # one block of M^-1 against the full-lattice oracle (block 0 and the last block, which touches the antiperiodic boundary)
    ora = OracleC(dims, Ls, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
    ora.load_gauge(Uabi, -1)
    z = g.unpack(g.apply_precond(g.pack(d, F32), k, F32, LAYOUT_NATIVE), F32)
    rows = gpu_rows(torch, z, Ls)
    nb = [L // B for L, B in zip(dims, block)]
    for bidx in (0, ora.num_blocks - 1):
        r = bidx
        bo = []
        for dd in range(4):
            bo.append((r % nb[dd]) * block[dd]); r //= nb[dd]
        xcb = block_xcb(cfg, bo)
        ref = ora.apply_precond(src, k, only_block=bidx).reshape(Ls, -1, 24)[:, xcb]
        got = rows(xcb)
        assert np.abs(ref).sum() > 0
        assert rel(got, ref) <= 2e-2, (bidx, rel(got, ref))
        assert site_max(got, ref) <= 0.1, (bidx, site_max(got, ref))
    del z, ora
    g.close()
    torch.cuda.empty_cache()
    # the fp16 sloppy outer operator (tile kernel on the FULL geometry)
    g2 = Mspcg(dims, Ls, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
    g2.configure(F16, F16, 18)
    g2.load_gauge(Uabi, -1)
    out16 = g2.unpack(g2.apply_MdagM(g2.pack(d, F16), F16, LAYOUT_NATIVE), F16)
    check_MdagM_windows(cfg, U, src, gpu_rows(torch, out16, Ls), origins, 2e-3, 1e-2)
    g2.close()


def rows_to_field(rows, loc, ext):
    """ABI rows [Ls, n, 4, 3, 2] on the box sites `loc` (x, y, z, t) -> oracle field psi[s, t, z, y, x, spin, colour] of the box."""
    f = np.zeros((rows.shape[0], ext[3], ext[2], ext[1], ext[0], 4, 3), dtype=np.complex128)
    f[:, loc[:, 3], loc[:, 2], loc[:, 1], loc[:, 0]] = rows[..., 0] + 1j * rows[..., 1]
    return f


def field_to_rows(f, loc):
    v = f[:, loc[:, 3], loc[:, 2], loc[:, 1], loc[:, 0]]
    return np.stack([v.real, v.imag], axis=-1)


def test_C4_reduced_Ls_preconditioner_one_block():
    """C4's reduced-Ls preconditioner (Ls 12 -> 6, eq. 20-21) on one 16^3 x 32 block, untrained T: eq. 20 composed by
    oracle/reduced_ls.py (ReducedLsPrecond, apply_T, apply_Tdag act per site, here on the block's sites) around the C oracle's
    Ls_hat block CG on the 2B-periodic lattice that reproduces the block and its pad (module docstring)."""
    from oracle import reduced_ls
    import torch
    cfg = synth.CONFIGS["C4"]
    dims, Ls, block, k, Lh, mu = cfg["dims"], cfg["Ls"], cfg["block"], 4, cfg["Ls_hat"], 0.85
    U = synth.random_su3_links(dims, cfg["eps"], cfg["gauge_seed"])
    src = synth.gaussian_spinor_abi(dims, Ls, cfg["src_seed"])
    T = reduced_ls.initial_T(Ls, Lh)
    g = Mspcg(dims, Ls, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
    g.set_reduced_ls(Lh, reduced_ls.T_to_abi(T), mu)
    g.configure(F32, F16, 18)
    g.load_gauge(synth.gauge_natural_to_abi(U, dims), -1)
    d = torch.as_tensor(src.reshape(-1)).cuda()
    z = g.unpack(g.apply_precond(g.pack(d, F32), k, F32, LAYOUT_NATIVE, use_reduced=1), F32)
    bo = (16, 0, 16, 32)
    xcb, loc = window_sites(dims, bo, block)
    got = gpu_rows(torch, z, Ls)(xcb)
    ext = tuple(2 * b for b in block)
    org = tuple(o - 2 for o in bo)
    sub = np.roll(cut_links(U, dims, org, ext), (-2, -2, -2, -2), axis=(4, 3, 2, 1))
    hatC = OracleC(ext, Lh, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
    hatC.load_gauge(synth.gauge_natural_to_abi(sub, ext), +1)
    xs, _ = window_sites(ext, (0, 0, 0, 0), block)

    def pre_hat(rh_field, kk):   # block CG at Ls_hat on block 0 of the small lattice
        sm = np.zeros((Lh, int(np.prod(ext)) // 2, 4, 3, 2))
        sm[:, xs] = field_to_rows(rh_field, loc)
        out = hatC.apply_precond(sm, kk, only_block=0).reshape(Lh, -1, 4, 3, 2)[:, xs]
        return rows_to_field(out, loc, block)

    r_field = rows_to_field(src[:, xcb], loc, block)
    ref = field_to_rows(reduced_ls.ReducedLsPrecond(pre_hat, T, mu)(r_field, k), loc).reshape(Ls, -1, 24)
    assert rel(got, ref) <= 2e-2 and site_max(got, ref) <= 0.1, (rel(got, ref), site_max(got, ref))
    g.close()


def _free_host_gib():
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable"):
                return int(line.split()[1]) / 2**20
    except OSError:
        pass
    return 0.0


def test_C5_largest_instance_12_real_links():
    """C5 (48^3 x 96, Ls 12, mf 0.001, 8^4 blocks, 12-real links, outer fp32 / inner fp16 with fp64 reliable updates): sloppy fp32 D^dag D
    windows (12-real links, third row rebuilt in the kernels) and the fp16-storage preconditioner of two blocks rebuilt on a 16^4 lattice."""
    if _free_host_gib() < 60:
        pytest.skip("C5 needs ~45 GiB of host memory for the links and the source in two layouts (have %.0f GiB)" % _free_host_gib())
    import torch
    cfg = synth.CONFIGS["C5"]
    dims, Ls, block, k = cfg["dims"], cfg["Ls"], cfg["block"], cfg["n_inner"]
    small = synth.random_su3_links((16, 16, 16, 32), cfg["eps"], cfg["gauge_seed"])
    U = np.tile(small, (1, 3, 3, 3, 3, 1, 1))
    del small
    g, U, Uabi, src, torch = make(cfg, F32, F16, recon=12, U_nat=U)
    del Uabi
    origins = [(2, 4, 6, 8), (dims[0] - 6, 2, 0, dims[3] - 6), (2, 2, 2, 2)]

    def native32():   # the workspace takes 153 of the 178 GiB: only one fp64 ABI vector (11.4 GiB) may live on the device at a time
        dd = torch.as_tensor(src.reshape(-1)).cuda()
        v = g.pack(dd, F32)
        del dd
        torch.cuda.empty_cache()
        return v

    def to_abi(nat):
        torch.cuda.empty_cache()
        return g.unpack(nat, F32)

    v32 = native32()
    q32 = g.apply_MdagM(v32, F32, LAYOUT_NATIVE)
    del v32
    out32 = to_abi(q32)
    del q32
    check_MdagM_windows(cfg, U, src, gpu_rows(torch, out32, Ls), origins, 1e-5, 1e-5)
    del out32
    torch.cuda.empty_cache()
    v32 = native32()
    z32 = g.apply_precond(v32, k, F32, LAYOUT_NATIVE)
    del v32
    z = to_abi(z32)
    del z32
    rows = gpu_rows(torch, z, Ls)
    ext = tuple(2 * b for b in block)
    for bo in ((0, 0, 0, 0), (40, 8, 16, 88)):     # the second block touches the antiperiodic time boundary
        xcb = block_xcb(cfg, bo)
        org = tuple(o - 2 for o in bo)
        sub = np.roll(cut_links(U, dims, org, ext), (-2, -2, -2, -2), axis=(4, 3, 2, 1))
        ora = OracleC(ext, Ls, cfg["b"], cfg["c"], cfg["M5"], cfg["mf"], block)
        ora.load_gauge(synth.gauge_natural_to_abi(sub, ext), +1)
        xs, _ = window_sites(ext, (0, 0, 0, 0), block)
        sm = np.zeros((Ls, int(np.prod(ext)) // 2, 4, 3, 2))
        sm[:, xs] = src[:, xcb]
        ref = ora.apply_precond(sm, k, only_block=0).reshape(Ls, -1, 24)[:, xs]
        got = rows(xcb)
        assert rel(got, ref) <= 2e-2 and site_max(got, ref) <= 0.1, (bo, rel(got, ref), site_max(got, ref))
    g.close()
