"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/mspcg.h declares, validates its
arguments, and its host-side tables (site sets, fifth-dimension matrices) agree with the paper-derived goldens.
No compute call is made (no GPU here)."""
import os
import re

import numpy as np
import pytest

from paper_2104_05615_b200 import Mspcg, MspcgError, binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "mspcg.h")).read()
    declared = set(re.findall(r"\b(mspcg_[a-zA-Z0-9_]+)\s*\(", hdr))
    declared -= {"mspcg_ctx"}
    assert declared == set(binding.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_create_validates_arguments(lib):
    ok = dict(dims=(4, 4, 4, 4), Ls=8, b=1.5, c=0.5, M5=1.8, mf=0.01, block=(2, 2, 2, 2))
    Mspcg(**ok).close()
    for bad in (dict(dims=(4, 4, 4, 5)), dict(block=(3, 2, 2, 2)), dict(block=(2, 2, 2, 8)), dict(Ls=1), dict(Ls=7),
                dict(b=-1.0 / 2.2, M5=1.8)):  # alpha = b(4-M5)+1 = 0
        kw = dict(ok)
        kw.update(bad)
        with pytest.raises(MspcgError):
            Mspcg(**kw)


def test_site_sets_match_golden_shell_counts(lib):
    """Minimal site sets of PAPER.md:226 (R11): |E0|, |O1|, |E2| from the shell counts of SURVEY 8(a) A7."""
    rows = [l.split() for l in open(os.path.join(ROOT, "tests", "golden", "shell_counts.txt")) if not l.startswith("#")]
    for Bx, By, Bz, Bt, interior, d1, d2 in [tuple(int(x) for x in r) for r in rows]:
        B = (Bx, By, Bz, Bt)
        m = Mspcg(tuple(2 * b for b in B), 8, 1.5, 0.5, 1.8, 0.01, B)
        g = m.geometry()
        assert g["nblk"] == 16 and g["vh"] == 16 * interior // 2
        assert g["nE0"] == interior // 2
        assert g["nO1"] == interior // 2 + d1 // 2          # odd sites, overshoot <= 1
        assert g["nE2"] == interior // 2 + d1 // 2 + d2 // 2  # even sites, overshoot <= 2
        m.close()


@pytest.mark.parametrize("dims,block", [((16, 16, 16, 32), (8, 8, 8, 8)), ((4, 4, 4, 4), (2, 2, 2, 2)), ((2, 4, 6, 6), (2, 2, 6, 2)),
                                        ((8, 4, 4, 6), (4, 4, 2, 6)), ((12, 12, 12, 12), (6, 6, 6, 12)), ((4, 6, 4, 4), (2, 6, 2, 2))])
def test_tile_tables_of_the_fp16_tile_kernel(lib, dims, block):
    """Host logic of hop_tile.cuh (tile_tables.hpp, the cell-ordered site lists of geometry.hpp): every output site of every stage list in
    exactly one tile, every neighbour reference resolved to the shared-memory slot that holds that neighbour, absent neighbours on the
    zero column, copy runs consecutive and complete -- on the C2 geometry, the wrap-around case L - B < 4, ragged and uncut directions.
    Reuse: a full 4x4x2x2 cell stages 4.0 input columns per output site instead of 8."""
    m = Mspcg(dims, 8, 1.5, 0.5, 1.8, 0.01, block)
    st = m.tile_check()
    g = m.geometry()
    assert st["tiles_k3k5"] >= -(-g["nE0"] // 32) and st["tiles_k4"] >= -(-g["nO1"] // 32)
    if dims == (16, 16, 16, 32):
        assert st["tiles_k3k5"] == 64 and st["inputs_per_output_k3k5"] == 4.0 and st["inputs_per_output_full"] == 4.0
        assert st["inputs_per_output_k4"] < 5.0
    m.close()


def test_uncut_direction_has_no_halo(lib):
    m = Mspcg((4, 4, 4, 8), 8, 1.5, 0.5, 1.8, 0.01, (4, 4, 4, 8))
    g = m.geometry()
    assert g["nblk"] == 1 and g["nE0"] == g["nE2"] == g["nO1"] == g["vh"]


def test_fifth_dimension_matrices(lib):
    """R3/R4: M5 = alpha + beta S_minus on P+, M5^-1 M5 = 1, first column vs the golden of SURVEY R4."""
    for Ls, mf in ((8, 0.01), (16, 0.002), (12, 0.005), (4, 0.3), (6, 1.0)):
        m = Mspcg((4, 4, 4, 4), Ls, 1.5, 0.5, 1.8, mf)
        A, F, Ai = m.matrix("m5"), m.matrix("mphi"), m.matrix("m5inv")
        alpha, beta = 1.5 * 2.2 + 1.0, 0.5 * 2.2 - 1.0
        S = np.diag(np.ones(Ls - 1), -1)
        S[0, Ls - 1] = -mf
        assert np.allclose(A, alpha * np.eye(Ls) + beta * S, atol=1e-15)
        assert np.allclose(F, -0.5 * (1.5 * np.eye(Ls) + 0.5 * S), atol=1e-15)
        assert np.abs(Ai @ A - np.eye(Ls)).max() < 1e-15
        m.close()
    gold = [float(l) for l in open(os.path.join(ROOT, "tests", "golden", "m5inv_first_column.txt")) if not l.startswith("#")]
    m = Mspcg((4, 4, 4, 4), 16, 1.5, 0.5, 1.8, 0.002)
    assert np.allclose(m.matrix("m5inv")[:5, 0], gold, rtol=1e-2)


def test_workspace_size_is_reported_without_a_gpu(lib):
    m = Mspcg((8, 8, 8, 8), 8, 1.5, 0.5, 1.8, 0.01, (4, 4, 4, 4))
    n16 = m.workspace_bytes(binding.F32, binding.F16, 18)
    m2 = Mspcg((8, 8, 8, 8), 8, 1.5, 0.5, 1.8, 0.01, (4, 4, 4, 4))
    n64 = m2.workspace_bytes(binding.F64, binding.F64, 18)
    assert 0 < n16 < n64
    with pytest.raises(MspcgError):
        m.workspace_bytes(3, 2, 18)


def test_product_has_no_oracle_import():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2104_05615_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f


def test_apply_calls_fail_loudly_without_workspace(lib):
    """Error behaviour stated in include/mspcg.h: compute entry points return an error code (never a CPU result) when
    the workspace has not been set; checked through the raw C ABI with dummy non-null pointers (nothing is dereferenced)."""
    import ctypes as C
    m = Mspcg((4, 4, 4, 4), 8, 1.5, 0.5, 1.8, 0.01, (2, 2, 2, 2))
    a, b = C.c_void_p(256), C.c_void_p(512)
    assert lib.mspcg_apply_M5inv(m.h, a, b, 0, None) != 0
    assert lib.mspcg_apply_MdagM(m.h, a, b, binding.F64, 0, None) != 0
    assert lib.mspcg_apply_precond(m.h, a, b, binding.F64, 0, 6, 0, None) != 0
    assert lib.mspcg_apply_M5inv(None, a, b, 0, None) != 0
    m.close()
