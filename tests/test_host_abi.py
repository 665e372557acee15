"""Host-side checks of the C ABI that need no GPU: the library loads, exports every symbol declared in
include/subcycle.h, validates hierarchy descriptions (nesting rules, S13/S20) and sizes the
arena. No compute calls."""
import ctypes as C
import os
import re

import pytest

import paper_2503_09629_b200 as sc
from paper_2503_09629_b200 import workloads as wl
from paper_2503_09629_b200.binding import (SC_ERR_INVALID_ARG, SC_ERR_NESTING, SC_ERR_UNSUPPORTED, SubcycleError)

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    from paper_2503_09629_b200 import build
    build.build()
    return sc.lib()


def test_exports_every_declared_symbol(built):
    hdr = open(os.path.join(ROOT, "include", "subcycle.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(sc_[a-z_]+)\s*\(", hdr)))
    assert declared and set(declared) == set(sc.EXPORTS)
    for name in declared:
        assert hasattr(built, name), name


def _bytes(w):
    d, keep = sc.make_desc(w.boxes, w.domain_cells, w.nfields, w.ghost, w.xlo, w.xhi, w.coupling)
    return sc.sc_arena_bytes(d)


def test_all_baseline_configs_validate_and_size(built):
    gib = 1 << 30
    sizes = {name: _bytes(w) / gib for name, w in
             (("cfg1", wl.cfg1()), ("cfg2", wl.cfg2(128)), ("cfg3", wl.cfg3()), ("cfg4", wl.cfg4()),
              ("cfg5", wl.cfg5()), ("ragged", wl.ragged_small()))}
    # 7 arrays per field and box (2 state slots x (u, rho) + Y2r, Y3r, Y4r) — half of
    # SURVEY 8(a)'s 14-array plan (cfg 3 ~ 1.0 GiB, cfg 5 ~ 11.3 GiB, cfg 4 ~ 18.7 GiB); cfg 4 adds 2 scratch
    # arrays per field for the coupling products
    assert 0.45 < sizes["cfg3"] < 0.7
    assert 5.2 < sizes["cfg5"] < 6.8
    assert 11.0 < sizes["cfg4"] < 15.0
    assert sizes["cfg5"] < 170  # fits one B200


def test_work_accounting_matches_survey(built):
    assert wl.cfg1().updates_per_coarse_step(True) == 98304
    assert wl.cfg1().updates_per_coarse_step(False) == 131072
    assert wl.cfg3().updates_per_coarse_step(True) == 31457280
    assert wl.cfg3().updates_per_coarse_step(False) == 67108864
    assert abs(wl.cfg4().updates_per_coarse_step(True) / 1.501e8 - 1) < 2e-3
    assert abs(wl.cfg4().updates_per_coarse_step(False) / 4.341e8 - 1) < 2e-3
    assert abs(wl.cfg5().updates_per_coarse_step(True) / 1.057e9 - 1) < 1e-3
    assert abs(wl.cfg5().updates_per_coarse_step(False) / 3.221e9 - 1) < 1e-3


def test_nesting_validator_rejects_bad_hierarchies(built):
    L = sc.lib()
    B = wl.Box

    def rc(boxes, dom=(32, 32, 32), **kw):
        d, keep = sc.make_desc(boxes, dom, **kw)
        out = C.c_void_p()
        r = L.sc_create_hierarchy(C.byref(d), C.byref(out))
        assert not out.value or r == 0
        if out.value:
            L.sc_destroy(out)
        return r, L.sc_last_error().decode()

    base = [B(0, (0, 0, 0), (32, 32, 32))]
    # config 4 as literally written (two 96^3 finest boxes at +-0.3 of the level-2 extent): not nested
    lit = wl.nested_cubes(6, 96)
    ext2 = 96 * 4 // 2
    off = int(0.3 * ext2) * 16
    c6 = 96 * 64 // 2
    lit += [B(6, (c6 - off - 48, c6 - 48, c6 - 48), (96, 96, 96)), B(6, (c6 + off - 48, c6 - 48, c6 - 48), (96, 96, 96))]
    assert rc(lit, (96, 96, 96))[0] == SC_ERR_NESTING
    assert rc(base + [B(1, (9, 16, 16), (16, 16, 16))])[0] == SC_ERR_NESTING       # odd lo
    assert rc(base + [B(1, (16, 16, 16), (15, 16, 16))])[0] == SC_ERR_NESTING      # odd n
    assert rc(base + [B(1, (6, 16, 16), (16, 16, 16))])[0] == SC_ERR_NESTING       # margin 3 < 4
    assert rc(base + [B(1, (8, 16, 16), (16, 16, 16))])[0] != SC_ERR_NESTING       # margin 4 ok
    # siblings: any distance is fine (they exchange ghosts, NEXT-2), interiors must not overlap
    assert rc(base + [B(1, (8, 8, 8), (16, 16, 16)), B(1, (30, 8, 8), (16, 16, 16))])[0] != SC_ERR_NESTING  # gap 6
    assert rc(base + [B(1, (8, 8, 8), (16, 16, 16)), B(1, (24, 8, 8), (16, 16, 16))])[0] != SC_ERR_NESTING  # abutting
    assert rc(base + [B(1, (8, 8, 8), (16, 16, 16)), B(1, (22, 8, 8), (16, 16, 16))])[0] == SC_ERR_NESTING  # overlap
    assert rc([B(0, (0, 0, 0), (32, 32, 16))])[0] == SC_ERR_NESTING                # level 0 must cover the domain
    assert rc(base + [B(2, (40, 40, 40), (16, 16, 16))], nlevels=3)[0] == SC_ERR_NESTING  # empty level 1
    assert rc(base, ref_ratio=4)[0] == SC_ERR_UNSUPPORTED
    assert rc(base, ghost=1)[0] == SC_ERR_UNSUPPORTED
    assert rc(base, ghost=6)[0] == SC_ERR_UNSUPPORTED
    assert rc(base, ghost=5)[0] != SC_ERR_UNSUPPORTED
    assert rc(base, fd_order=8)[0] == SC_ERR_UNSUPPORTED            # 8th-order differences read 4 ghost layers
    assert rc(base, fd_order=6)[0] == SC_ERR_UNSUPPORTED
    assert rc(base, ghost=4, fd_order=8, ko_sigma=0.1)[0] == SC_ERR_UNSUPPORTED   # eq 36 with r = 8: delta^10 reads 5 layers
    assert rc(base, ghost=4, fd_order=8, ko_sigma=0.1, ko_order=5)[0] != SC_ERR_UNSUPPORTED  # the paper's production pair
    assert rc(base, ghost=5, fd_order=8, ko_sigma=0.1)[0] != SC_ERR_UNSUPPORTED
    assert rc(base, ghost=4, fd_order=8)[0] != SC_ERR_UNSUPPORTED
    # NEXT-3 / NEXT-4 options
    assert rc(base, integrator=5)[0] == SC_ERR_UNSUPPORTED
    assert rc(base, integrator=3)[0] != SC_ERR_UNSUPPORTED and rc(base, integrator=2)[0] != SC_ERR_UNSUPPORTED
    assert rc(base, outer_bc=2)[0] == SC_ERR_UNSUPPORTED
    assert rc(base, outer_bc=1, xlo=(0.5, -1.0, -1.0), xhi=(2.0, 1.0, 1.0))[0] == SC_ERR_INVALID_ARG  # origin outside
    # ... or inside the boundary zone of `ghost` points at a face, where the operator evaluates 1/r (dx0 = 3/32, g = 3)
    r_, msg_ = rc(base, outer_bc=1, xlo=(-0.25, -1.0, -1.0), xhi=(2.75, 1.0, 1.0))
    assert r_ == SC_ERR_INVALID_ARG and "1/r" in msg_
    assert rc(base, outer_bc=1, xlo=(-0.3, -1.0, -1.0), xhi=(2.7, 1.0, 1.0))[0] != SC_ERR_INVALID_ARG
    assert rc(base, ko_order=7)[0] == SC_ERR_UNSUPPORTED
    assert rc(base, interp=1)[0] == SC_ERR_UNSUPPORTED              # the 10-point restriction reads 4 ghost layers
    assert rc(base, interp=1, ghost=4)[0] != SC_ERR_UNSUPPORTED
    assert rc(base + [B(1, (8, 16, 16), (16, 16, 16))], vertex=1)[0] == SC_ERR_NESTING   # vertex: margin 5
    assert rc(base + [B(1, (10, 16, 16), (12, 16, 16))], vertex=1)[0] != SC_ERR_NESTING
    assert rc(base + [B(1, (10, 16, 16), (12, 16, 16))], interp=1, ghost=4)[0] == SC_ERR_NESTING  # 9-point: margin 6
    assert rc(base + [B(1, (12, 16, 16), (8, 16, 16))], interp=1, ghost=4)[0] != SC_ERR_NESTING
    assert rc(base, nfields=0)[0] == SC_ERR_UNSUPPORTED
    assert rc(base, xlo=(1.0, -1.0, -1.0), xhi=(1.0, 1.0, 1.0))[0] == SC_ERR_INVALID_ARG
    r, msg = rc(base + [B(1, (6, 16, 16), (16, 16, 16))])
    assert "margin" in msg or "parent" in msg


def test_null_and_range_errors_do_not_abort(built):
    L = sc.lib()
    assert L.sc_arena_bytes(None) == 0
    assert L.sc_create_hierarchy(None, None) == SC_ERR_INVALID_ARG
    assert L.sc_step(None, 0.1, 1) == SC_ERR_INVALID_ARG
    assert L.sc_set_state(None, 0, 0, 0, None, 0) == SC_ERR_INVALID_ARG
    assert L.sc_read_level(None, 0, 0, 0, None, 0) == SC_ERR_INVALID_ARG
    assert L.sc_destroy(None) == 0
    assert L.sc_time(None) == 0.0


def test_dissipation_in_the_description(built):
    """ko_sigma (eqs 35-36): validated on the host, and it buys 5 more arrays per field (U2..U4, k_4)."""
    w = wl.cfg3(n=32, nlevels=3)
    base = _bytes(w)
    d, keep = sc.make_desc(w.boxes, w.domain_cells, w.nfields, w.ghost, w.xlo, w.xhi, w.coupling, ko_sigma=0.2)
    with_ko = sc.sc_arena_bytes(d)
    assert with_ko > base and abs(with_ko / base - 12.0 / 7.0) < 0.01
    for bad in (-0.1, float("nan"), float("inf")):
        d, keep = sc.make_desc(w.boxes, w.domain_cells, ko_sigma=bad)
        assert sc.lib().sc_arena_bytes(d) == 0
    d, keep = sc.make_desc(w.boxes, w.domain_cells, ghost=2, ko_sigma=0.1)   # Q reads 3 ghost layers
    assert sc.lib().sc_arena_bytes(d) == 0
    assert b"ghost" in sc.lib().sc_last_error()


def _golden_rationals():
    from fractions import Fraction
    rows = {}
    for name in ("interp_weights.txt", "interp_weights_next.txt"):
        for line in open(os.path.join(ROOT, "tests", "golden", name)):
            if line.strip() and not line.startswith("#"):
                t = line.split()
                rows[t[0]] = [Fraction(x) for x in t[1:]]
    return rows


def test_product_interpolation_weights_are_the_correctly_rounded_rationals(built):
    """The LIBRARY's own prolongation / restriction operators (sc_debug_interp_weights; csrc/hierarchy.cpp derives them
    in exact integer arithmetic) against the rational tables under tests/golden/ — the 5-/6-point rows are SURVEY 8(c)'s,
    the 6-/9-/10-point rows come from make_interp_rationals.py (python fractions; neither oracle nor library) — and the
    tables themselves against what defines them: exactness on monomials up to degree np - 1 at the geometric position of
    the target, and NOT one degree more. float(Fraction) is correctly rounded, and so must the library's value be: ==."""
    from fractions import Fraction as Fr
    g = _golden_rationals()
    cases = {  # (interp, vertex) -> (prolong parity-1 row, its target, restriction row)
        (0, 0): ("prolong1", Fr(1, 4), "restrict"), (1, 0): ("prolong9_p1", Fr(1, 4), "restrict10"),
        (0, 1): ("vertex6_mid", Fr(1, 2), None), (1, 1): ("vertex10_mid", Fr(1, 2), None)}
    for (interp, vertex), (prow, x, rrow) in cases.items():
        P = sc.sc_debug_interp_weights(interp, vertex)
        assert not P["tail"].any()
        w1 = g[prow]
        assert P["np"] == len(w1) and [float(v) for v in w1] == list(P["w"][1])
        nodes = [Fr(P["pmin"] + m) for m in range(P["np"])]
        for k in range(P["np"] + 1):  # the rationals are the interpolation weights at x: exact to degree np - 1 only
            assert (sum(w * xm ** k for w, xm in zip(w1, nodes)) == x ** k) == (k < P["np"])
        if vertex:      # fine point 2J sits on parent point J: copy; restriction is injection
            assert list(P["w"][0]) == [1.0 if P["pmin"] + m == 0 else 0.0 for m in range(P["np"])]
            assert P["nr"] == 1 and P["rmin"] == 0 and list(P["r"]) == [1.0]
            assert P["pmin"] == -(P["np"] // 2 - 1)
        else:           # parity 0 is the mirror image about parent cell 0
            assert list(P["w"][0]) == list(P["w"][1])[::-1] and P["pmin"] == -(P["np"] // 2)
            r = g[rrow]
            assert P["nr"] == len(r) and [float(v) for v in r] == list(P["r"])
            fine = [Fr(2 * (P["rmin"] + m) - 1, 2) for m in range(P["nr"])]  # centre of fine cell 2I + j: j - 1/2 from the parent centre
            assert fine[0] == -fine[-1]
            for k in range(P["nr"] + 1):
                # symmetric stencil: odd monomials vanish identically, so "one degree more" is tested on even k only
                ok = sum(w * xm ** k for w, xm in zip(r, fine)) == (1 if k == 0 else 0)
                assert ok == (k < P["nr"] or k % 2 == 1)
    L = sc.lib()
    assert L.sc_debug_interp_weights(2, 0, None, None, None, None, None, None, None) == sc.binding.SC_ERR_UNSUPPORTED
