"""The C-ABI boundary without a GPU: liblbm.so loads, exports every symbol include/lbm.h declares,
validates its arguments on the host, reports the lattice tables the kernels use, and refuses to run
without a CUDA device (no CPU fallback).  No compute call is made here.  `-m "not gpu"`."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lbm():
    import __graft_entry__ as ge
    ge.build()                       # nvcc cross-compiles for sm_100a without a GPU
    import paper_2502_12955_b200 as pkg
    pkg.lib()
    return pkg


def declared_symbols():
    """function names declared in include/lbm.h"""
    src = open(os.path.join(ROOT, "include", "lbm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lbm_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lbm):
    names = declared_symbols()
    assert "lbm_create" in names and "lbm_step" in names and "lbm_get_macros" in names
    assert "lbm_init_from_seed" in names and "lbm_destroy" in names
    L = lbm.lib()
    for n in names:
        assert hasattr(L, n), "liblbm.so does not export %s" % n
    assert sorted(lbm.SYMBOLS) == names          # the binding lists exactly the header's functions


def test_params_struct_matches_header(lbm):
    """struct_size is checked by the library: a ctypes layout that disagreed with the C struct would
    make every call fail with 'struct_size'."""
    p = lbm.make_params(**workloads.config("cfg4")["params"])
    n = lbm.lib().lbm_workspace_bytes(256, 256, 256, lbm.D3Q19, lbm.BGK, C.byref(p))
    assert n >= 19 * 256 ** 3 * 8 and n < 19 * 256 ** 3 * 8 + 4096     # ONE population copy, no psi
    p.struct_size -= 8
    assert lbm.lib().lbm_workspace_bytes(256, 256, 256, lbm.D3Q19, lbm.BGK, C.byref(p)) == 0
    assert "struct_size" in lbm.lbm.last_error()


@pytest.mark.parametrize("name,expect", [
    ("cfg1", 9 * 8), ("cfg2", (9 + 1) * 8), ("cfg3", (18 + 2) * 8), ("cfg4", 19 * 8), ("cfg5", (38 + 7 + 2) * 4)])
def test_workspace_is_one_population_copy_plus_psi(lbm, name, expect):
    """in-place streaming: S*Q + Qs values per cell and S values of psi, nothing else"""
    cfg = workloads.config(name)
    p = lbm.make_params(**cfg["params"])
    nx, ny, nz = cfg["grid"]
    n = lbm.lib().lbm_workspace_bytes(nx, ny, nz, lbm.lbm.LATTICES[cfg["lattice"]], lbm.lbm.MODELS[cfg["model"]], C.byref(p))
    N = nx * ny * nz
    assert expect * N <= n <= expect * N + 3 * 256


@pytest.mark.parametrize("grid,lattice,model,over,msg", [
    ((8, 8, 2), "D2Q9", "BGK", {}, "nz == 1"),
    ((8, 8, 8), "D3Q19", "BGK", dict(tau=(0.5, 0.5)), "tau"),
    ((8, 8, 8), "D3Q19", "BGK", dict(precision=16), "precision"),
    ((8, 8, 8), "D3Q19", "SC2_ADE", dict(tau_c=0.4, bc=(0, 0, 0)), "tau_c"),
    ((0, 8, 8), "D3Q19", "BGK", {}, "extents"),
    ((2048, 2048, 1024), "D3Q19", "BGK", {}, "2^31"),
    ((8, 8, 8), "D3Q19", "BGK", dict(forcing=2), "forcing"),
    ((1024, 1024, 512), "D3Q19", "BGK", {}, "2^32"),
    ((8, 8, 8), "D3Q19", "SC2", dict(psi_kind=2, bc=(0, 0, 0)), "psi_kind"),
    ((8, 8, 8), "D3Q19", "SC1", dict(psi_kind=0, rho0_psi=0.0, bc=(0, 0, 0)), "rho0_psi"),
    ((8, 8, 1), "D2Q9", "BGK", dict(bc=(0, 0, 1)), "bc[2]"),
])
def test_validation_messages(lbm, grid, lattice, model, over, msg):
    p = lbm.make_params(**dict(workloads.config("cfg4")["params"], **over))
    n = lbm.lib().lbm_workspace_bytes(grid[0], grid[1], grid[2], lbm.lbm.LATTICES[lattice], lbm.lbm.MODELS[model], C.byref(p))
    assert n == 0
    assert msg in lbm.lbm.last_error()


def test_null_arguments_are_errors_not_crashes(lbm):
    L = lbm.lib()
    assert L.lbm_step(None, 1) == lbm.lbm.EINVAL
    assert L.lbm_init_from_seed(None, 0) == lbm.lbm.EINVAL
    assert L.lbm_get_macros(None, None, None, None, None) == lbm.lbm.EINVAL
    assert L.lbm_population_count(None) == 0
    assert L.lbm_time(None) == -1 and L.lbm_launch_count(None) == -1
    L.lbm_destroy(None)
    assert L.lbm_workspace_bytes(8, 8, 8, 1, 0, None) == 0


def test_lattice_tables_of_the_kernels_match_the_paper(lbm):
    """lbm_lattice_table (the compile-time tables the kernels unroll over) against the paper's
    Tables 1-3 stored in tests/golden/lattice_tables.txt (w_4 of D2Q9: R1)."""
    from fractions import Fraction
    blocks, cur = {}, None
    for line in open(os.path.join(ROOT, "tests", "golden", "lattice_tables.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("["):
            cur = line[1:-1]
            blocks[cur] = {}
        else:
            k, *v = line.split()
            blocks[cur][k] = v
    for name, lattice, kind in [("D3Q19", "D3Q19", 0), ("D2Q9", "D2Q9", 0), ("D2Q5", "D2Q9", 1)]:
        c, w, opp = lbm.lattice_table(lattice, kind)
        b = blocks[name]
        assert len(w) == len(b["w"])
        assert np.allclose(w, [float(Fraction(x)) for x in b["w"]], rtol=0, atol=1e-16)
        assert list(c[:, 0]) == [int(x) for x in b["cx"]]
        assert list(c[:, 1]) == [int(x) for x in b["cy"]]
        if "cz" in b:
            assert list(c[:, 2]) == [int(x) for x in b["cz"]]
        for i in range(len(w)):
            assert (c[opp[i]] == -c[i]).all()
        assert abs(w.sum() - 1) < 1e-15
    c, w, opp = lbm.lattice_table("D3Q19", 1)          # D3Q7 (R6)
    assert len(w) == 7 and w[0] == 0.25 and np.all(w[1:] == 0.125)
    assert [tuple(r) for r in c[1:]] == [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]


def test_no_cpu_fallback(lbm):
    """Without a CUDA device lbm_create must fail loudly (and the binding must not route elsewhere)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    p = lbm.make_params(**workloads.config("cfg1")["params"])
    h = lbm.lib().lbm_create(8, 8, 1, lbm.D2Q9, lbm.BGK, C.byref(p))
    assert not h
    assert "no usable CUDA device" in lbm.lbm.last_error() and "no CPU path" in lbm.lbm.last_error()
    with pytest.raises(lbm.LbmError):
        lbm.LBM(8, 8, 1, "D2Q9", "BGK")


def test_product_path_never_touches_the_oracle():
    """Neither the package nor the C/CUDA sources mention oracle/ or ref_lbm (independence of the two paths)."""
    pkg = os.path.join(ROOT, "paper_2502_12955_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "ref_lbm" not in text and "import oracle" not in text and "from oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "liblbm" not in text and "kernels.cuh" not in text and "import paper_2502_12955_b200" not in text, f


@pytest.mark.parametrize("nm,ns,py", [(1, 1, 1), (1, 7, 1), (1, 64, 1), (5, 4, 2), (8, 8, 3), (8, 8, 8), (2, 2, 1), (3, 1, 2),
                                      (16, 9, 5), (6, 5, 100), (40, 12, 7)])
@pytest.mark.parametrize("wrap_m,wrap_s", [(True, True), (False, True), (True, False), (False, False)])
@pytest.mark.parametrize("delay", [0, 3])
def test_tile_schedule_is_valid(nm, ns, py, wrap_m, wrap_s, delay):
    """Host logic of the resident-tile kernel (tile_schedule.h).  Every row has exactly one STEP item (pencil order)
    and exactly one PSI item (psi of the next time level, R9).  A PSI item needs the step of the 3 x 3 rows around
    its row (periodic wrap or wall; Eq. 5 / 7): it is listed exactly `delay` STEP rows after the LAST of their STEP
    items (or at the very end) -- never before (the block that takes it would wait for a later step), never later
    than asked (the populations would leave L2) -- so the PSI items are ordered by the time they become ready.  Rows
    that wait for another pencil or for the wrapped plane are re-read from HBM: they must stay a small fraction."""
    import paper_2502_12955_b200 as pkg
    it, deferred = pkg.lbm.tile_schedule(nm, ns, py, wrap_m, wrap_s, delay)
    assert len(it) == 2 * nm * ns
    step_pos, psi_pos = {}, {}
    for k, (kind, m, s) in enumerate(it.tolist()):
        assert kind in (0, 1) and 0 <= m < nm and 0 <= s < ns
        d = step_pos if kind == 0 else psi_pos
        assert (m, s) not in d
        d[(m, s)] = k
    assert len(step_pos) == nm * ns and len(psi_pos) == nm * ns
    p = max(1, min(py, nm))
    steps = [(m, s) for kind, m, s in it.tolist() if kind == 0]
    assert steps == [(m, s) for m0 in range(0, nm, p) for s in range(ns) for m in range(m0, min(m0 + p, nm))]
    order = {ms: k for k, ms in enumerate(steps)}
    late = 0
    for (m, s), k in psi_pos.items():
        deps = []
        for dm in (-1, 0, 1):
            for ds in (-1, 0, 1):
                mm, ss = m + dm, s + ds
                if (not wrap_m and not 0 <= mm < nm) or (not wrap_s and not 0 <= ss < ns):
                    continue
                deps.append(step_pos[(mm % nm, ss % ns)])
        last = max(deps)
        assert last < k                                   # after its last dependency ...
        between = sum(1 for kind, _, _ in it[last + 1:k].tolist() if kind == 0)
        assert between == delay or (between < delay and all(kind == 1 for kind, _, _ in it[k:].tolist()))     # ... by `delay` step rows
        if max(order[(it[d][1], it[d][2])] for d in deps) - order[(m, s)] > 2 * p + 8:
            late += 1
    assert late == deferred
    pencils = -(-nm // p)
    assert deferred <= pencils * (2 * ns + 2 * (p + 2)) + 2




@pytest.mark.parametrize("nm,ns,nxs,py,delay,three_d", [(1, 9, 3, 1, 0, False), (1, 40, 2, 1, 5, False), (6, 5, 2, 2, 0, True),
                                                        (8, 7, 3, 3, 4, True), (5, 4, 1, 8, 2, True), (1, 1, 1, 1, 0, True),
                                                        (12, 10, 2, 4, 30, True)])
@pytest.mark.parametrize("wrap_m,wrap_s", [(True, True), (False, True), (True, False), (False, False)])
def test_tile_tickets_depend_only_on_earlier_tickets(nm, ns, nxs, py, delay, three_d, wrap_m, wrap_s):
    """The tickets the resident-tile kernel deals out round-robin (tile_schedule.h tile_tickets, used by lbm_set_path):
    every tile is stepped by exactly one ticket and has its psi formed by exactly one ticket; the psi part of ticket k
    reads what the steps of the (up to 27) tiles around its tile have written, and each of those steps is the step part
    of a ticket with a SMALLER index -- with blocks that take their tickets in order and are all resident, the earliest
    unfinished ticket can therefore always proceed; the tail of psi-only tickets stays short."""
    import paper_2502_12955_b200 as pkg
    tk = pkg.lbm.tile_tickets(nm, ns, nxs, py, wrap_m, wrap_s, delay, three_d).tolist()
    n_tiles = nm * ns * nxs
    step_at, psi_at = {}, {}
    for k, (sx, sy, sz, sv, px, py_, pz, pv) in enumerate(tk):
        assert sv or pv
        if sv:
            assert (sx, sy, sz) not in step_at and 0 <= sx < nxs
            step_at[(sx, sy, sz)] = k
        if pv:
            assert (px, py_, pz) not in psi_at and 0 <= px < nxs
            psi_at[(px, py_, pz)] = k
    assert len(step_at) == n_tiles and len(psi_at) == n_tiles
    assert all(tk[k][3] for k in range(n_tiles))                 # the first n_tiles tickets all step
    def rows_around(y, z):
        m, s = (y, z) if three_d else (0, y)
        for dm in (-1, 0, 1):
            for ds in (-1, 0, 1):
                mm, ss = m + dm, s + ds
                if (not wrap_m and not 0 <= mm < nm) or (not wrap_s and not 0 <= ss < ns):
                    continue
                mm, ss = mm % nm, ss % ns
                yield (mm, ss) if three_d else (ss, 0)
    for (px, y, z), k in psi_at.items():
        for (yy, zz) in rows_around(y, z):
            for dx in (-1, 0, 1):
                assert step_at[((px + dx) % nxs, yy, zz)] < k
    p = max(1, min(py, nm))
    # tail: the rows that only the LAST pencil completes (its own last planes, the wrapped plane, the columns of rows
    # beside it) and the delay -- a vanishing fraction of a large grid
    assert len(tk) - n_tiles <= (2 * ns + 3 * (p + 2) + delay) * nxs + 1
