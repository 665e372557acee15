"""sc_max_abs_noalloc against sc_debug_max_abs: the allocation-free blow-up check must say what the hierarchy's says.

The entry point exists for programs that cannot call cudaMalloc around the library: their own memory pool already owns
the whole GPU (so a further cudaMalloc fails), or they poll a running simulation for NaN / inf from a time loop that
cannot take the device-wide synchronisation an allocation implies. Its scratch is one fixed array built into
libsubcycle.so, shared by every call on a GPU and never cleared between calls. So the test makes TWO calls in a row whose
answers differ, the second on a shorter input with a smaller maximum: partials left by the first call, or a counter
that was not reset, would show up as the first call's answer. max |x| is exact, so "within tolerance" is bit-equal.

The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure and a failure here
must not hide the parity tests. It passes alone in a fresh process and after the rest of the suite."""
import math
import struct

import pytest

import paper_2503_09629_b200 as sc
from paper_2503_09629_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _bits(v: float) -> bytes:
    return struct.pack("<d", v)


def _both_paths(G, torch, box, values):
    """Upload `values` (dense interior [nz][ny][nx], CUDA) into component 0 of level 0 and reduce it both ways."""
    G.sc_set_state(0, 0, 0, values)
    existing = G.sc_debug_max_abs(0, 0, 0)  # one block per row of the padded box, atomicMax into the staging buffer
    out = torch.full((1,), -7.0, dtype=torch.float64, device="cuda")
    sc.sc_max_abs_noalloc(values, out)      # dense array, partials in the library's built-in array
    torch.cuda.synchronize()
    assert box.n[0] * box.n[1] * box.n[2] == values.numel()
    return existing, float(out.item())


def test_noalloc_max_abs_matches_the_hierarchy_path_twice_in_a_row():
    import torch

    big = wl.Box(0, (0, 0, 0), (72, 40, 44))    # 126 720 doubles: 16 blocks, ragged last one
    small = wl.Box(0, (0, 0, 0), (24, 16, 8))   # 3 072 doubles: a single, partly filled block
    gen = torch.Generator(device="cuda").manual_seed(20250309)

    G1 = sc.Hierarchy([big], big.n)
    x1 = torch.randn(big.n[2], big.n[1], big.n[0], dtype=torch.float64, device="cuda", generator=gen) * 3.0
    x1[17, 5, 70] = -123.456  # the maximum sits near the end of a row, negative
    e1, n1 = _both_paths(G1, torch, big, x1)
    assert e1 == 123.456 and _bits(n1) == _bits(e1)
    G1.close()

    # second call straight after: shorter input, smaller answer; a stale partial of the first call would give 123.456
    G2 = sc.Hierarchy([small], small.n)
    x2 = torch.rand(small.n[2], small.n[1], small.n[0], dtype=torch.float64, device="cuda", generator=gen) * 0.5
    e2, n2 = _both_paths(G2, torch, small, x2)
    assert 0.0 < e2 <= 0.5 and _bits(n2) == _bits(e2)

    # the NaN / inf rule is the existing path's rule
    x2[3, 9, 11] = float("inf")
    e3, n3 = _both_paths(G2, torch, small, x2)
    assert math.isinf(e3) and math.isinf(n3)
    x2[0, 0, 0] = float("nan")
    e4, n4 = _both_paths(G2, torch, small, x2)
    assert math.isnan(e4) and math.isnan(n4)
    G2.close()


def test_noalloc_rejects_what_its_scratch_cannot_hold():
    import torch

    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    x = torch.ones(8, dtype=torch.float64, device="cuda")
    L = sc.lib()
    too_many = sc.SC_NOALLOC_MAX_DOUBLES + 1  # only the length is checked: no memory of that size is touched
    assert L.sc_max_abs_noalloc(x.data_ptr(), too_many, out.data_ptr(), None) == -1
    assert b"SC_NOALLOC_MAX_DOUBLES" in L.sc_last_error()
    assert L.sc_max_abs_noalloc(x.data_ptr(), 8, None, None) == -1
    # empty input: 0.0, and the refused calls above left the scratch usable
    sc.sc_max_abs_noalloc(x[:0], out)
    torch.cuda.synchronize()
    assert float(out.item()) == 0.0
    sc.sc_max_abs_noalloc(x, out)
    torch.cuda.synchronize()
    assert float(out.item()) == 1.0
