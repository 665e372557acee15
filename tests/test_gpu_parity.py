"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerance (BASELINE.json north_star, reading S27): u components max|delta| <= 1e-11 * max|u|, rho components
<= 1e-11 * max|rho| + the rounding floor of the definition, ghosts included (oracle/parity.py is the one statement);
index maps and the set_state -> read_level round trip bit-exact. Run on the B200 box with `-m gpu`."""
import numpy as np
import pytest

import oracle
import paper_2503_09629_b200 as sc
from oracle.parity import RTOL, compare_state as _compare_state  # the one statement of the tolerance
from paper_2503_09629_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _pair(w):
    return sc.Hierarchy.from_workload(w), oracle.OracleHierarchy.from_workload(w)


def test_set_read_roundtrip_bit_exact():
    w = wl.ragged_small()
    G = sc.Hierarchy.from_workload(w)
    for l in range(w.nlevels):
        for ib in range(len(w.level_boxes(l))):
            for c in range(w.ncomp):
                assert np.array_equal(G.sc_read_level(l, ib, c), w.initial_state(l, ib, c))
    # device-side source and destination
    import torch
    src = torch.arange(40 * 24 * 28, dtype=torch.float64, device="cuda").reshape(28, 24, 40) * 0.5
    G.sc_set_state(0, 0, 1, src)
    out = torch.empty_like(src)
    G.sc_read_level(0, 0, 1, out)
    assert torch.equal(out, src)
    G.close()


def test_ghost_index_map_bit_exact():
    w = wl.ragged_small()
    G, O = _pair(w)
    for l in (1, 2):
        for ib in range(len(w.level_boxes(l))):
            assert np.array_equal(G.sc_debug_ghost_map(l, ib), O.ghost_map(l, ib))
    w = wl.cfg4(n=32, nlevels=4, nfields=1)
    G2, O2 = sc.Hierarchy(w.boxes, w.domain_cells), oracle.OracleHierarchy(w.boxes, w.domain_cells)
    for ib in (0, 1):
        assert np.array_equal(G2.sc_debug_ghost_map(3, ib), O2.ghost_map(3, ib))


def test_single_level_step_and_slopes():
    """One periodic level: rhs + stage combine + periodic fill alone; also k_1..k_4 and y_old."""
    w = wl.Workload("t", [wl.Box(0, (0, 0, 0), (40, 24, 28))], (40, 24, 28), nfields=2,
                    coupling=wl.coupling_matrix(2), init=wl.multi_gaussian_init(3))
    G, O = _pair(w)
    for sub in (True, False, True):
        G.sc_step(w.dt_coarse, sub)
        O.step(w.dt_coarse, sub)
        _compare_state(G, O, w, what=f"single level sub={sub}")
    _compare_stored_stages(G, O, w, 0, 0, w.dt_coarse, y4=False)


def _compare_stored_stages(G, O, w, level, ib, dt, y4=True):
    """What the CUDA path keeps of a level-step (S26): y_n and the rho-parts of Y_2, Y_3, Y_4, against
    the oracle's y_old and Y_{s+1,rho} = rho_n + a_s dt k_{s,rho} (eqs 7-9) built from its stored slopes.
    Y_4's rho-part (= k_{4,u}) is stored only on levels whose child reads it (subcycled mode)."""
    F = w.nfields
    for c in range(w.ncomp):
        a, b = G.sc_debug_read_slot(level, ib, 1, c), O.read(level, ib, c, slot=O.SLOT_YOLD)
        assert np.max(np.abs(a - b)) <= RTOL * max(np.max(np.abs(b)), 1e-300), ("y_n", c)
    for s, a_s in ((2, 0.5), (3, 0.5), (4, 1.0))[:3 if y4 else 2]:
        for f in range(F):
            b = O.read(level, ib, F + f, slot=O.SLOT_YOLD) + a_s * dt * O.read(level, ib, F + f, slot=O.SLOT_K1 + s - 2)
            a = G.sc_debug_read_slot(level, ib, s, F + f)
            assert np.max(np.abs(a - b)) <= RTOL * max(np.max(np.abs(b)), 1e-300), (s, f)
    with pytest.raises(sc.SubcycleError):
        G.sc_debug_read_slot(level, ib, 2, 0)  # the u-part of a stage vector is never stored


@pytest.mark.parametrize("sub", [True, False])
def test_two_level_one_step_ghosts_slopes_restriction(sub):
    """After ONE coarse step: ghosts of both levels (stage-5 fill), parent cells under the child
    (restriction), child slopes."""
    w = wl.cfg1()
    G, O = _pair(w)
    G.sc_step(w.dt_coarse, sub)
    O.step(w.dt_coarse, sub)
    _compare_state(G, O, w, what=f"cfg1 one step sub={sub}")
    if sub:
        _compare_stored_stages(G, O, w, 0, 0, w.dt_coarse)
        _compare_stored_stages(G, O, w, 1, 0, w.dt_coarse / 2, y4=False)


@pytest.mark.parametrize("sub", [True, False])
def test_cfg1_full_run(sub):
    w = wl.cfg1()
    G, O = _pair(w)
    for _ in range(w.coarse_steps):
        G.sc_step(w.dt_coarse, sub)
        O.step(w.dt_coarse, sub)
    rel = _compare_state(G, O, w, what=f"cfg1 8 steps sub={sub}")
    assert abs(G.sc_time() - O.time) < 1e-15
    print(f"cfg1 sub={sub}: max rel diff {rel:.2e}")


@pytest.mark.parametrize("sub", [True, False])
def test_ragged_multibox_coupled(sub):
    """Non-cubic boxes, ragged tile tails, two sibling boxes on the finest level, F = 2 with coupling."""
    w = wl.ragged_small()
    G, O = _pair(w)
    for _ in range(3):
        G.sc_step(w.dt_coarse, sub)
        O.step(w.dt_coarse, sub)
        _compare_state(G, O, w, what=f"ragged sub={sub}")


@pytest.mark.parametrize("sub", [True, False])
def test_cfg3_shape_scaled(sub):
    """4 nested levels (config 3 shape) at 48^3, 3 coarse steps."""
    w = wl.cfg3(n=48, nlevels=4)
    G, O = _pair(w)
    for _ in range(3):
        G.sc_step(w.dt_coarse, sub)
        O.step(w.dt_coarse, sub)
    _compare_state(G, O, w, what=f"cfg3/48 sub={sub}")


def test_cfg4_shape_scaled():
    """BBH-shaped (config 4): 5 levels of 32^3, finest = two boxes, 6 coupled fields, 2 coarse steps."""
    w = wl.cfg4(n=32, nlevels=5, nfields=6)
    G, O = _pair(w)
    for sub in (True, False):
        G.sc_step(w.dt_coarse, sub)
        O.step(w.dt_coarse, sub)
        _compare_state(G, O, w, what=f"cfg4/32 sub={sub}")


@pytest.mark.parametrize("sub", [True, False])
def test_cfg5_full_depth_reduced_n(sub):
    """cfg 5's level count (6 nested levels) at 64^3: every level, ghosts included, after two coarse steps. Deep
    recursion element by element: theta = 1/2 fills prefilled on the side branch of the graph (levels this small
    take it), Y4r kept on levels 2..4, every state-slot phase combination of the graph key."""
    w = wl.cfg5(64, 6)
    G, O = _pair(w)
    for _ in range(2):
        G.sc_step(w.dt_coarse, sub)
        O.step(w.dt_coarse, sub)
    rel = _compare_state(G, O, w, what=f"cfg5/64 x6 sub={sub}")
    print(f"cfg5 64^3 x 6 levels sub={sub}: max|d|/max|u| = {rel:.2e}")
    G.close()


def test_cfg4_full_depth_reduced_n():
    """cfg 4's level count (7 levels, the finest = two boxes) and all 22 coupled fields at 32^3, one subcycled step."""
    w = wl.cfg4(32, 7, 22)
    G, O = _pair(w)
    G.sc_step(w.dt_coarse, True)
    O.step(w.dt_coarse, True)
    rel = _compare_state(G, O, w, what="cfg4/32 x7 F=22")
    print(f"cfg4 32^3 x 7 levels, 22 fields: max|d|/max|u| = {rel:.2e}")
    G.close()


def test_cfg2_rung_matches_oracle_and_exact_solution():
    """Config 2, 32^3 rung to t = 1 (64 coarse steps): parity and the error against the exact plane wave."""
    w = wl.cfg2(32)
    G, O = _pair(w)
    for _ in range(w.coarse_steps):
        G.sc_step(w.dt_coarse, True)
        O.step(w.dt_coarse, True)
    _compare_state(G, O, w, what="cfg2/32")
    for l in (0, 1):
        err = np.max(np.abs(G.sc_read_level(l, 0, 0) - wl.plane_wave_exact(w, l, 0, 0, 1.0)))
        assert 5.5e-5 < err < 7e-5, (l, err)


def test_ghost_width_2_and_4():
    for g in (2, 4):
        w = wl.cfg1()
        w.ghost = g
        G, O = _pair(w)
        G.sc_step(w.dt_coarse, True)
        O.step(w.dt_coarse, True)
        _compare_state(G, O, w, what=f"ghost={g}")


def test_graph_replay_equals_eager(monkeypatch):
    """CUDA-graph replay (default) and plain stream launches (SC_GRAPH=0) give identical bits."""
    w = wl.cfg3(n=32, nlevels=3)
    G1 = sc.Hierarchy.from_workload(w)
    monkeypatch.setenv("SC_GRAPH", "0")
    G2 = sc.Hierarchy.from_workload(w)
    monkeypatch.delenv("SC_GRAPH")
    for _ in range(3):
        G1.sc_step(w.dt_coarse, True)
        G2.sc_step(w.dt_coarse, True)
    for l in range(3):
        for c in range(2):
            assert np.array_equal(G1.sc_debug_read_padded(l, 0, c), G2.sc_debug_read_padded(l, 0, c))
    assert G1.sc_launch_count() == G2.sc_launch_count() > 0


def test_varying_dt_updates_the_graph_in_place(monkeypatch):
    """An adaptive-dt caller: 300 coarse steps with 300 distinct step sizes, modes alternating. The executable graphs are
    keyed by (mode, slot phase) only; a new dt re-records the launches and updates the existing executable in place:
    a handful of instantiations, a bounded cache, no growth of device memory, and the same bits as eager launches."""
    import torch
    w = wl.ragged_small()
    G1 = sc.Hierarchy.from_workload(w)
    monkeypatch.setenv("SC_GRAPH", "0")
    G2 = sc.Hierarchy.from_workload(w)
    monkeypatch.delenv("SC_GRAPH")
    free0 = None
    for i in range(300):
        dt = w.dt_coarse * (0.5 + 0.001 * i)
        sub = (i // 3) % 2 == 0
        G1.sc_step(dt, sub)
        G2.sc_step(dt, sub)
        if i == 20:
            G1.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
    G1.synchronize()
    st = G1.sc_debug_graph_stats()
    assert st["instantiations"] <= 8 and st["cached"] <= 8, st
    assert st["updates"] >= 280 and st["captures"] == st["updates"] + st["instantiations"], st
    assert torch.cuda.mem_get_info()[0] >= free0 - (8 << 20), (free0, torch.cuda.mem_get_info()[0])
    for l in range(w.nlevels):
        for ib in range(len(w.level_boxes(l))):
            for c in range(w.ncomp):
                assert np.array_equal(G1.sc_debug_read_padded(l, ib, c), G2.sc_debug_read_padded(l, ib, c))
    assert G2.sc_debug_graph_stats()["captures"] == 0
    # the same dt again: pure replay
    G1.sc_step(w.dt_coarse, True)
    G1.sc_step(w.dt_coarse, True)
    G1.sc_step(w.dt_coarse, True)
    st2 = G1.sc_debug_graph_stats()
    assert st2["captures"] <= st["captures"] + 2, (st, st2)


def test_error_paths_on_device():
    w = wl.cfg1()
    G = sc.Hierarchy.from_workload(w)
    with pytest.raises(sc.SubcycleError):
        G.sc_step(float("nan"))
    with pytest.raises(sc.SubcycleError):
        G.sc_step(-1.0)
    with pytest.raises(sc.SubcycleError):
        G.sc_read_level(5, 0, 0)
    with pytest.raises(sc.SubcycleError):
        G.sc_debug_ghost_map(0, 0)
    G.sc_step(w.dt_coarse)  # still usable afterwards
    G.close()


@pytest.mark.parametrize("g", [2, 3, 4])
def test_ghost_fill_geometry_sweep(g):
    """Child boxes at every offset class (lo mod 4 per axis decides tile origins, footprint parity and the
    alignment of every TMA coordinate), sizes that are not multiples of any tile, inside parents whose padded
    extent the last footprints overrun: one subcycled + one uniform step each, every ghost and interior value."""
    B = wl.Box
    cases = [
        ((40, 24, 28), (10, 8, 12), (32, 32, 26)),   # odd parent x index of the first footprint cell
        ((64, 64, 64), (22, 20, 20), (44, 28, 26)),
        ((64, 64, 64), (20, 22, 26), (30, 46, 18)),
        ((48, 40, 36), (8, 8, 8), (66, 50, 42)),     # child reaches the nesting margin on the high sides
        ((36, 36, 36), (14, 18, 10), (20, 14, 34)),
        ((32, 32, 32), (8, 8, 8), (48, 48, 48)),
    ]
    for dom, lo, n in cases:
        w = wl.Workload(f"sweep {dom} {lo} {n} g={g}", [B(0, (0, 0, 0), dom), B(1, lo, n)], dom, ghost=g,
                        init=wl.multi_gaussian_init(3))
        G, O = _pair(w)
        for sub in (True, False):
            G.sc_step(w.dt_coarse, sub)
            O.step(w.dt_coarse, sub)
            _compare_state(G, O, w, what=w.name + f" sub={sub}")
        assert np.array_equal(G.sc_debug_ghost_map(1, 0), O.ghost_map(1, 0))
        G.close()


@pytest.mark.parametrize("sub", [True, False])
def test_exact_quadratic_solution_without_the_oracle(sub):
    """The CUDA path against a closed form, no oracle involved: u = x^2+y^2+z^2+3t^2, rho = 6t is reproduced
    exactly by every operator of the scheme (see tests/test_oracle_scheme.py), so after one coarse step of a
    3-level hierarchy every level must hold it to rounding away from level 0's periodic seam."""
    n = 64
    w = wl.Workload("quadratic", wl.nested_cubes(3, n), (n, n, n), init=wl.quadratic_init)
    G = sc.Hierarchy.from_workload(w)
    G.sc_step(w.dt_coarse, sub)
    t = w.dt_coarse
    for l in (1, 2):
        for c in (0, 1):
            got = G.sc_debug_read_padded(l, 0, c)
            want = wl.quadratic_exact(w, l, 0, c, t, pad=w.ghost)
            assert np.max(np.abs(got - want)) < 2e-12, (sub, l, c, float(np.max(np.abs(got - want))))
    m = slice(10, n - 10)
    for c in (0, 1):
        assert np.max(np.abs(G.sc_read_level(0, 0, c)[m, m, m] - wl.quadratic_exact(w, 0, 0, c, t)[m, m, m])) < 2e-12
    G.close()


# ---- NEXT-1: Kreiss-Oliger dissipation (eqs 35-36), general stage-by-stage path -------------------
def _with_ko(w, sigma=0.25):
    w.ko_sigma = sigma
    w.name += f" + KO sigma={sigma}"
    return w


@pytest.mark.parametrize("sub", [True, False])
def test_ko_cfg1_full_run(sub):
    w = _with_ko(wl.cfg1())
    G, O = _pair(w)
    for _ in range(w.coarse_steps):
        G.sc_step(w.dt_coarse, sub)
        O.step(w.dt_coarse, sub)
    rel = _compare_state(G, O, w, what=f"KO cfg1 sub={sub}")
    print(f"KO cfg1 sub={sub}: max rel diff {rel:.2e}")
    # the dissipation did something: the undamped run differs by far more than the tolerance
    G0 = sc.Hierarchy.from_workload(wl.cfg1())
    for _ in range(w.coarse_steps):
        G0.sc_step(w.dt_coarse, sub)
    assert np.max(np.abs(G0.sc_read_level(1, 0, 0) - G.sc_read_level(1, 0, 0))) > 1e-8


@pytest.mark.parametrize("sub", [True, False])
def test_ko_ragged_multibox_coupled(sub):
    w = _with_ko(wl.ragged_small(), 0.1)
    G, O = _pair(w)
    for _ in range(3):
        G.sc_step(w.dt_coarse, sub)
        O.step(w.dt_coarse, sub)
        _compare_state(G, O, w, what=f"KO ragged sub={sub}")


def test_ko_four_levels_and_mode_switch():
    w = _with_ko(wl.cfg3(n=48, nlevels=4), 0.3)
    G, O = _pair(w)
    for sub in (True, False, True):
        G.sc_step(w.dt_coarse, sub)
        O.step(w.dt_coarse, sub)
    _compare_state(G, O, w, what="KO cfg3/48")


@pytest.mark.parametrize("sub", [True, False])
def test_ko_exact_quadratic_solution_without_the_oracle(sub):
    n = 64
    w = wl.Workload("quadratic+KO", wl.nested_cubes(3, n), (n, n, n), init=wl.quadratic_init, ko_sigma=0.2)
    G = sc.Hierarchy.from_workload(w)
    G.sc_step(w.dt_coarse, sub)
    t = w.dt_coarse
    for l in (1, 2):
        for c in (0, 1):
            got = G.sc_debug_read_padded(l, 0, c)
            assert np.max(np.abs(got - wl.quadratic_exact(w, l, 0, c, t, pad=w.ghost))) < 5e-12, (sub, l, c)
    m = slice(14, n - 14)
    for c in (0, 1):
        assert np.max(np.abs(G.sc_read_level(0, 0, c)[m, m, m] - wl.quadratic_exact(w, 0, 0, c, t)[m, m, m])) < 5e-12
    G.close()


def test_ko_needs_three_ghost_layers():
    w = wl.cfg1()
    w.ghost = 2
    w.ko_sigma = 0.1
    with pytest.raises(sc.SubcycleError):
        sc.Hierarchy.from_workload(w)


# ---- NEXT-2: same-level ghost exchange between sibling boxes (kernels.h a7) -------------------------------------
SIB_CUTS = {"x halves": ((24,), (), ()), "z 8+16": ((), (), (20,)), "quarters + near box": ((24,), (22,), ()),
            "eight boxes": ((24,), (20,), (20,))}


@pytest.mark.parametrize("sigma", [0.0, 0.2])
@pytest.mark.parametrize("sub", [True, False])
def test_sibling_exchange_parity(sub, sigma):
    """Abutting, edge-touching and near (2 cells apart) level-1 boxes, 2 coupled fields: CUDA path vs oracle,
    ghosts included (a ghost cell inside a sibling holds the sibling's value)."""
    for name, (cx, cy, cz) in SIB_CUTS.items():
        w = wl.sibling_cut(cx, cy, cz, nfields=2, ko_sigma=sigma, near="near" in name)
        G, O = _pair(w)
        for _ in range(w.coarse_steps):
            G.sc_step(w.dt_coarse, sub)
            O.step(w.dt_coarse, sub)
        _compare_state(G, O, w, what=f"siblings {name} sub={sub} sigma={sigma}")
        G.close()


@pytest.mark.parametrize("sigma", [0.0, 0.2])
@pytest.mark.parametrize("sub", [True, False])
def test_cut_level_reproduces_the_uncut_level_on_the_gpu(sub, sigma):
    """Decomposition invariance without the oracle: a cell update reads the same numbers whether its neighbour
    lives in the same box or arrives through the exchange, so the cut level must match the uncut one to rounding
    (not bit for bit: the z-march accumulates the stencil's z terms in march order, which depends on where a
    cell sits in its box's z-chunks)."""
    def run(cuts):
        w = wl.sibling_cut(*cuts, ko_sigma=sigma)
        G = sc.Hierarchy.from_workload(w)
        for _ in range(3):
            G.sc_step(w.dt_coarse, sub)
        l1 = np.full((24, 24, 24), np.nan)
        for ib, b in enumerate(w.level_boxes(1)):
            o = [b.lo[a] - 12 for a in range(3)]
            l1[o[2]:o[2] + b.n[2], o[1]:o[1] + b.n[1], o[0]:o[0] + b.n[0]] = G.sc_read_level(1, ib, 0)
        out = (G.sc_read_level(0, 0, 0), l1, G.sc_read_level(2, 0, 0))
        G.close()
        return out
    ref = run(((), (), ()))
    for name, cuts in SIB_CUTS.items():
        got = run(cuts)
        for l in range(3):
            assert np.max(np.abs(got[l] - ref[l])) <= 1e-13 * np.max(np.abs(ref[l])), (name, l)


@pytest.mark.parametrize("sigma", [0.0, 0.2])
@pytest.mark.parametrize("sub", [True, False])
def test_exact_quadratic_solution_through_siblings_without_the_oracle(sub, sigma):
    """Closed form, no oracle: u = x^2+y^2+z^2+3t^2, rho = 6t through level-1 boxes that abut on a face, touch
    along an edge, or sit two cells apart; every box, ghosts included, must hold it to rounding."""
    n, o = 64, 16
    l1 = [wl.Box(1, (24 + o, 24 + o, 24 + o), (16, 24, 24)), wl.Box(1, (40 + o, 24 + o, 24 + o), (16, 24, 24)),
          wl.Box(1, (56 + o, 48 + o, 24 + o), (12, 16, 24)), wl.Box(1, (24 + o, 50 + o, 24 + o), (30, 14, 24))]
    boxes = [wl.Box(0, (0, 0, 0), (n, n, n))] + l1 + [wl.Box(2, (88 + 2 * o, 60 + 2 * o, 60 + 2 * o), (16, 16, 16))]
    w = wl.Workload("quadratic siblings", boxes, (n, n, n), init=wl.quadratic_init, ko_sigma=sigma)
    G = sc.Hierarchy.from_workload(w)
    G.sc_step(w.dt_coarse, sub)
    t = w.dt_coarse
    for l in (1, 2):
        for ib in range(len(w.level_boxes(l))):
            for c in (0, 1):
                got = G.sc_debug_read_padded(l, ib, c)
                want = wl.quadratic_exact(w, l, ib, c, t, pad=w.ghost)
                assert np.max(np.abs(got - want)) < 3e-12, (sub, l, ib, c, float(np.max(np.abs(got - want))))
    G.close()


# ---- the paper's own validation run (Fig. 1) --------------------------------------------------
def test_paper_fig1_ladder_on_the_gpu():
    """Gaussian spherical wave (eqs 41-42), three levels (r = 4, 1, 0.5), h_1 = 1/8, h_1/1.5, h_1/2, to t = 1.5
    (the pulse has crossed both refinement boundaries): fourth-order convergence of the error on the second
    refinement level against the exact solution, subcycled and uniform — no oracle involved; then parity with the
    oracle on the low resolution."""
    T = 1.5
    err = {}
    for sub in (True, False):
        for n0 in (64, 96, 128):
            w = wl.paper_wave(n0)
            G = sc.Hierarchy.from_workload(w)
            ns = int(round(T / w.dt_coarse))
            for _ in range(ns):
                G.sc_step(w.dt_coarse, sub)
            err[(sub, n0)] = max(np.max(np.abs(G.sc_read_level(2, 0, c) - wl.spherical_wave_exact(w, 2, 0, c, T)))
                                 for c in (0, 1))
            G.close()
        o1 = np.log(err[(sub, 64)] / err[(sub, 96)]) / np.log(1.5)
        o2 = np.log(err[(sub, 64)] / err[(sub, 128)]) / np.log(2.0)
        print(f"Fig. 1 on the GPU, sub={sub}: errors {err[(sub, 64)]:.3e} {err[(sub, 96)]:.3e} {err[(sub, 128)]:.3e}, orders {o1:.2f} {o2:.2f}")
        assert 3.7 < o1 < 4.3 and 3.7 < o2 < 4.3
    for n0 in (64, 96, 128):
        assert abs(err[(True, n0)] / err[(False, n0)] - 1.0) < 0.05
    w = wl.paper_wave(64)
    G, O = _pair(w)
    for _ in range(8):
        G.sc_step(w.dt_coarse, True)
        O.step(w.dt_coarse, True)
    _compare_state(G, O, w, what="paper Fig. 1, 8 subcycled steps")


def test_cfg2_convergence_ladder_on_the_gpu():
    """BASELINE config 2 as stated, whole and without the oracle: coarse 32^3, 64^3, 128^3 (fine boxes scaled to
    match), plane wave evolved to t = 1 (64 / 128 / 256 coarse steps); error against the exact solution on both
    levels, convergence order, both modes; and the subcycled - uniform difference, which must stay below the
    truncation error and itself converge (third order: eq (10)'s local error, DESIGN S12)."""
    err, sol = {}, {}
    for sub in (True, False):
        for n in (32, 64, 128):
            w = wl.cfg2(n)
            G = sc.Hierarchy.from_workload(w)
            for _ in range(w.coarse_steps):
                G.sc_step(w.dt_coarse, sub)
            assert abs(G.sc_time() - 1.0) < 1e-12
            sol[(sub, n)] = [G.sc_read_level(l, 0, 0) for l in (0, 1)]
            err[(sub, n)] = [float(np.max(np.abs(sol[(sub, n)][l] - wl.plane_wave_exact(w, l, 0, 0, 1.0)))) for l in (0, 1)]
            G.close()
        for l in (0, 1):
            o1 = np.log2(err[(sub, 32)][l] / err[(sub, 64)][l])
            o2 = np.log2(err[(sub, 64)][l] / err[(sub, 128)][l])
            print(f"cfg2 sub={sub} level {l}: errors {err[(sub, 32)][l]:.3e} {err[(sub, 64)][l]:.3e} {err[(sub, 128)][l]:.3e} orders {o1:.2f} {o2:.2f}")
            assert 3.8 < o1 < 4.2 and 3.8 < o2 < 4.2
    diff = [max(float(np.max(np.abs(a - b))) for a, b in zip(sol[(True, n)], sol[(False, n)])) for n in (32, 64, 128)]
    print("cfg2 max|sub - uniform|:", ["%.2e" % d for d in diff])
    for d, n in zip(diff, (32, 64, 128)):
        assert d < 0.5 * err[(True, n)][1]
    assert 2.5 < np.log2(diff[0] / diff[1]) < 4.5 and 2.5 < np.log2(diff[1] / diff[2]) < 4.5


def test_debug_max_abs():
    """sc_debug_max_abs: device-side max |x| over the interior; NaN as soon as one value is NaN, inf if one is
    infinite — the check for a run that blew up, without copying the state."""
    w = wl.ragged_small()
    G = sc.Hierarchy.from_workload(w)
    for l in range(w.nlevels):
        for ib in range(len(w.level_boxes(l))):
            for c in range(w.ncomp):
                assert G.sc_debug_max_abs(l, ib, c) == float(np.max(np.abs(w.initial_state(l, ib, c))))
    a = w.initial_state(1, 0, 0).copy()
    a[3, 5, 7] = np.inf
    G.sc_set_state(1, 0, 0, a)
    assert G.sc_debug_max_abs(1, 0, 0) == np.inf
    a[2, 1, 0] = np.nan
    G.sc_set_state(1, 0, 0, a)
    assert np.isnan(G.sc_debug_max_abs(1, 0, 0))
    G.close()


# ---- NEXT-3: 8th-order centred differences on the plain stage kernel ----------------------------
def _fd8(w):
    w.ghost, w.fd_order = 4, 8
    w.name += " + 8th-order FD"
    return w


@pytest.mark.parametrize("sub", [True, False])
def test_fd8_parity(sub):
    """cfg 1 (8 steps) and the ragged coupled multi-box hierarchy with 8th-order differences (ghost width 4)."""
    for w in (_fd8(wl.cfg1()), _fd8(wl.ragged_small())):
        G, O = _pair(w)
        for _ in range(w.coarse_steps):
            G.sc_step(w.dt_coarse, sub)
            O.step(w.dt_coarse, sub)
        _compare_state(G, O, w, what=f"{w.name} sub={sub}")
        G.close()


def test_fd8_closed_forms_without_the_oracle():
    """The CUDA path against closed forms: the exact quadratic solution through 3 levels, and the one-level plane
    wave whose error is RK4's omega T (omega dt)^4 / 120 once the differences are 8th order."""
    n = 64
    w = wl.Workload("quadratic fd8", wl.nested_cubes(3, n), (n, n, n), init=wl.quadratic_init, ghost=4, fd_order=8)
    G = sc.Hierarchy.from_workload(w)
    G.sc_step(w.dt_coarse, True)
    for l in (1, 2):
        for c in (0, 1):
            got = G.sc_debug_read_padded(l, 0, c)
            assert np.max(np.abs(got - wl.quadratic_exact(w, l, 0, c, w.dt_coarse, pad=4))) < 5e-12, (l, c)
    G.close()
    base = wl.cfg2(32)
    one = wl.Workload("one level fd8", base.boxes[:1], base.domain_cells, init=wl.plane_wave_init, ghost=4, fd_order=8)
    G = sc.Hierarchy.from_workload(one)
    for _ in range(base.coarse_steps):
        G.sc_step(one.dt_coarse, True)
    om = np.sqrt(3.0) * np.pi
    model = om * (om * one.dt_coarse) ** 4 / 120.0
    e = np.max(np.abs(G.sc_read_level(0, 0, 0) - wl.plane_wave_exact(one, 0, 0, 0, 1.0)))
    assert 0.7 * model < e < 1.3 * model, (e, model)
    G.close()


def test_fd8_needs_four_ghost_layers():
    w = wl.cfg1()
    with pytest.raises(sc.SubcycleError):
        sc.Hierarchy(w.boxes, w.domain_cells, ghost=3, fd_order=8)
    with pytest.raises(sc.SubcycleError):  # eq 36 with r = 8 reads 5 layers
        sc.Hierarchy(w.boxes, w.domain_cells, ghost=4, fd_order=8, ko_sigma=0.1)
