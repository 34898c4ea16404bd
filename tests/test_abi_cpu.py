"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/gmg.h declares; the Python binding names match; argument validation that needs no
GPU.  No compute calls here."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "gmg.h")


def _declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gmg_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2607_07687_b200 import build
    return build.build()


def test_header_declares_the_north_star_entry_points():
    syms = _declared_symbols()
    for name in ("gmg_create", "gmg_set_coeffs", "gmg_solve", "gmg_stats"):
        assert name in syms


def test_library_exports_every_declared_symbol(libpath):
    dll = C.CDLL(libpath)
    for name in _declared_symbols():
        assert hasattr(dll, name), f"{name} declared in gmg.h but not exported"
    out = subprocess.check_output(["nm", "-D", "--defined-only", libpath]).decode()
    exported = set(re.findall(r" T (gmg_[a-z0-9_]+)", out))
    assert exported == set(_declared_symbols())


def test_binding_covers_every_symbol(libpath):
    from paper_2607_07687_b200 import gmg
    assert sorted(gmg.SIGNATURES) == _declared_symbols()


def test_library_contains_sm100a_code(libpath):
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_struct_sizes_match_header(libpath):
    """Params / Stats mirror the C structs (17 x 4 bytes; Stats has 8-byte alignment)."""
    from paper_2607_07687_b200 import gmg
    assert C.sizeof(gmg.Params) == 68
    assert C.sizeof(gmg.Stats) == 4 * 4 + 6 * 8 + 8 + 8 + 3 * 8
    p = gmg.Params()
    gmg.lib.gmg_default_params(C.byref(p))
    assert (p.nu_pre, p.nu_post, p.nu_coarse, p.n_min) == (2, 2, 32, 4)
    assert (p.omega0, p.omega_min, p.omega_down, p.omega_up) == (1.0, 0.5, 0.125, 0.03125)
    assert (p.fast_path, p.use_graph, p.cluster_tail, p.fused_norm, p.uniform_tiles, p.small_cg) == (1, 1, 1, 1, 1, 1)


def test_null_arguments_are_rejected_without_a_gpu(libpath):
    from paper_2607_07687_b200 import gmg
    I3 = C.c_int * 3
    assert gmg.lib.gmg_create(None, 8, 8, 8, I3(0, 0, 0)) == gmg.EINVAL
    h = C.c_void_p()
    assert gmg.lib.gmg_create(C.byref(h), 7, 8, 8, I3(0, 0, 0)) == gmg.EINVAL   # odd periodic
    assert gmg.lib.gmg_create(C.byref(h), 0, 8, 8, I3(1, 0, 0)) == gmg.EINVAL   # extent < 1
    assert gmg.lib.gmg_create(C.byref(h), 8, 8, 1, I3(0, 0, 0)) == gmg.EINVAL   # extent 1 needs walls
    assert gmg.lib.gmg_create(C.byref(h), 8, 8, 8, I3(0, 2, 0)) == gmg.EINVAL   # bad bc
    assert gmg.lib.gmg_num_levels(None) == gmg.EINVAL
    assert gmg.lib.gmg_workspace_bytes(None) == 0


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_07687_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import oracle|from oracle)", txt, flags=re.M), f
                assert "gmg_oracle" not in txt and "libgmg_oracle" not in txt, f


# ---- host logic of the library, no GPU: level table (reading O4), tail choice, workspace size ----
def test_library_level_table_matches_golden_and_oracle(libpath):
    import oracle
    from paper_2607_07687_b200 import gmg
    gold = os.path.join(ROOT, "tests", "golden", "level_shapes.txt")
    for line in open(gold):
        if line.startswith("#") or not line.strip():
            continue
        name, bc, shapes = [s.strip() for s in line.split("|")]
        bc = tuple(int(x) for x in bc.split())
        shapes = [tuple(int(x) for x in s.split("x")) for s in shapes.split()]
        got, factors, tail, ws = gmg.plan(shapes[0], bc)
        assert got == shapes, name
        assert factors[-1] == (1, 1, 1)
        for l in range(len(shapes) - 1):
            assert tuple(a // f for a, f in zip(shapes[l], factors[l])) == shapes[l + 1]
        # the tail is a suffix whose 8 floats per cell fit 200 KB of shared memory
        cells = sum(s[0] * s[1] * s[2] for s in shapes[tail:])
        assert tail < len(shapes) and cells * 32 <= 200 * 1024
        assert tail == 0 or (cells + shapes[tail - 1][0] * shapes[tail - 1][1] * shapes[tail - 1][2]) * 32 > 200 * 1024
        # workspace: coarse levels (L, p, b, q) + level-0 q + 6 fine vectors + the six face weights
        # of the tail levels, each array 256-byte aligned; the cluster tail may take the weights of
        # levels above the single-CTA tail too (at most 32768 cells each)
        N = [s[0] * s[1] * s[2] for s in shapes]
        lower = 4 * (N[0] + 6 * N[0] + sum(6 * v for v in N[1:]) + sum(6 * v for v in N[tail:]))
        cluster_extra = 4 * sum(6 * v for v in N[:tail] if v <= 32768)
        # ... and one array as large as the largest TMA-fed level with 2x2x2 coarsening: the corrected
        # copy of the non-lean tiles for the sweep that folds the prolongation in (uniform.cuh)
        scratch = 4 * max([N[l] for l in range(min(tail, len(N) - 1))
                           if shapes[l][0] >= 128 and shapes[l][0] % 128 == 0 and factors[l] == (2, 2, 2)] + [0])
        assert lower <= ws <= lower + cluster_extra + scratch + 256 * (7 * len(N) + 9)
        if shapes[0] == (1024, 1024, 1024):
            assert ws >= lower + scratch
    # agreement with the oracle's rule on odd / mixed cases, both coarsening modes
    for n, bc in [((20, 20, 20), (1, 0, 0)), ((36, 20, 6), (0, 1, 0)), ((64, 4, 4), (1, 0, 0)), ((15, 9, 7), (1, 1, 1)),
                  ((64, 16, 1), (1, 0, 1)), ((128, 32, 1), (0, 0, 1))]:      # 2-D mode
        for iso in (False, True):
            got = gmg.plan(n, bc, coarsen_mode=gmg.COARSEN_ISO if iso else gmg.COARSEN_ANISO)[0]
            assert got == oracle.level_shapes(n, bc, iso=iso), (n, bc, iso)
    with pytest.raises(ValueError):
        gmg.plan((31, 32, 16), (0, 0, 0))


def test_jellyfish_step_sequence_is_compatible_and_moves_smoothly():
    """Input recipe of the warm-started pressure steps (S4): div u* sums to zero, solid
    cells carry no flux, and consecutive steps differ by a fraction of a cell of body motion."""
    import numpy as np
    from paper_2607_07687_b200 import workloads as W
    steps = list(W.jellyfish_steps(4, 4))
    assert len(steps) == 4
    prev = None
    for L, u in steps:
        assert L.dtype == np.float32 and u.dtype == np.float32 and L.shape == u.shape == (3, 16, 32, 32)
        assert L.min() >= 0.0 and L.max() <= 1.0 and (L == 0.0).any()
        z = W.divergence(u.astype(np.float64), W.JELLYFISH_BC)
        assert abs(z.sum()) < 1e-9 * np.abs(z).sum()
        act = W.active_mask(L, W.JELLYFISH_BC)
        assert np.all(z[~act] == 0.0)
        if prev is not None:
            assert 0.0 < np.abs(L - prev).max() < 0.5
        prev = L


def test_maximum_grid_size_is_planned_on_the_host_and_one_more_cell_is_refused(libpath):
    """The library indexes a level with 32-bit cell counts: 2^31 - 1 cells at most.  The largest
    grids are planned without a GPU (level table, workspace) and the first one too large is refused
    by gmg_plan and gmg_create alike."""
    from paper_2607_07687_b200 import gmg
    shapes, factors, tail, ws = gmg.plan((2048, 1024, 1022), (0, 0, 0))
    import oracle
    # periodic z: 1022 / 2 = 511 is odd, so z never coarsens (reading O4); x and y go down to 4
    assert shapes[0] == (2048, 1024, 1022) and shapes[1] == (1024, 512, 1022) and shapes[-1] == (4, 4, 1022)
    assert shapes == oracle.level_shapes((2048, 1024, 1022), (0, 0, 0))
    N = [s[0] * s[1] * s[2] for s in shapes]
    assert N[0] < 2 ** 31 and ws > 4 * 7 * N[0]
    with pytest.raises(ValueError):
        gmg.plan((2048, 1024, 1024), (0, 0, 0))                                  # 2^31 cells
    h = C.c_void_p()
    I3 = C.c_int * 3
    assert gmg.lib.gmg_create(C.byref(h), 2048, 1024, 1024, I3(0, 0, 0)) == gmg.EINVAL
