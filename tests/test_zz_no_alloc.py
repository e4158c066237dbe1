"""md_velocity_sums_noalloc (include/md_b200.h): the velocity sums of md_energies from a static device
scratch array -- an entry point that allocates nothing, for callers that cannot call cudaMalloc.  Checked against the
existing path (md_energies of an md_system, same velocities) on calls in a row that share the scratch array.

This file sorts last on purpose (pytest collects test files by name): the suite runs with `pytest -x`."""
import numpy as np
import pytest

from md_workloads import get_config, make_state
from parity_util import ENERGY_RTOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def md():
    import paper_2003_14061_b200 as m
    m.load_library()
    return m


def _check(md, g, out):
    """One call on the system's current velocities against md_energies.  `out`: a caller-owned device tensor, so that nothing
    -- neither the library nor the binding -- allocates inside the call."""
    import torch
    v = g.velocities_device()
    torch.cuda.synchronize()
    got = md.velocity_sums_noalloc(v, out=out)
    assert got.data_ptr() == out.data_ptr()
    torch.cuda.synchronize()
    ke, px, py, pz, vmax = out.cpu().numpy()
    e = g.energies()
    assert ke == pytest.approx(e.ke, rel=ENERGY_RTOL)
    scale = np.sqrt(2.0 * e.ke * g.n)                        # sum |v_i| <= sqrt(2 ke N): the size of the terms the momentum sums
    for a, b in ((px, e.px), (py, e.py), (pz, e.pz)):
        assert abs(a - b) <= 1e-12 * scale + 1e-12
    assert vmax == pytest.approx(e.vmax, rel=1e-12)
    # and against the definition, from the host copy of the same array
    vh = v.cpu().numpy()
    assert ke == pytest.approx(0.5 * float((vh * vh).sum()), rel=1e-12)
    assert vmax == pytest.approx(float(np.sqrt((vh * vh).sum(1).max())), rel=1e-14)
    return np.array([ke, px, py, pz, vmax])


def test_two_calls_in_a_row_equal_md_energies(md):
    import torch
    out = torch.full((5,), float("nan"), dtype=torch.float64, device="cuda")
    # a large system first (2048 blocks of partials), then a small ragged one (5 blocks): the second call finds the first
    # call's partials in the shared scratch array and must not read them
    big = get_config("wca_2m")
    gb = md.MDSystem(big.n_atoms, big.r_cut, big.r_shell, big.dt, density=big.density)
    gb.step(5)
    first = _check(md, gb, out)
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 3, jitter_amp=0.1)
    n = 4097 - 96                                                # not a multiple of the block's 1024 atoms, nor of 32
    gs = md.MDSystem(n, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    gs.set_state(r[:n], v[:n] + 0.01)                            # a net momentum: the sums are not all ~0
    second = _check(md, gs, out)
    assert abs(second[1]) > 1.0 and second[0] < 1e-2 * first[0]
    # the same input again: bitwise the same result (fixed summation order), and again after the state moved on
    third = _check(md, gs, out)
    assert np.array_equal(second, third)
    gs.step(40)
    fourth = _check(md, gs, out)
    assert not np.array_equal(third, fourth)
    again = _check(md, gb, out)                                  # back to the large system
    assert np.array_equal(first, again)
    gb.close()
    gs.close()


def test_single_precision_state_and_one_atom(md):
    """The boundary arrays are binary64 in both precisions, so the entry point serves a binary32 system too; n = 1."""
    import torch
    cfg = get_config("wca_4k")
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, density=cfg.density, precision="f32")
    g.step(20)
    out = torch.empty(5, dtype=torch.float64, device="cuda")
    _check(md, g, out)
    g.close()
    one = torch.tensor([[3.0, -4.0, 12.0]], dtype=torch.float64, device="cuda")
    md.velocity_sums_noalloc(one, out=out)
    assert out.cpu().numpy().tolist() == [84.5, 3.0, -4.0, 12.0, 13.0]


def test_rejects_what_it_cannot_hold(md):
    import ctypes as C
    import torch
    L = md.load_library()
    v = torch.zeros((8, 3), dtype=torch.float64, device="cuda")
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    host = np.zeros((8, 3))
    too_many = md.NOALLOC_MAX_ATOMS + 1
    assert L.md_velocity_sums_noalloc(C.c_void_p(v.data_ptr()), too_many, C.c_void_p(out.data_ptr()), None) == -1
    assert b"MD_NOALLOC_MAX_ATOMS" in L.md_last_error()
    assert L.md_velocity_sums_noalloc(C.c_void_p(v.data_ptr()), 0, C.c_void_p(out.data_ptr()), None) == -1
    assert L.md_velocity_sums_noalloc(C.c_void_p(host.ctypes.data), 8, C.c_void_p(out.data_ptr()), None) == -1
    assert L.md_velocity_sums_noalloc(C.c_void_p(v.data_ptr()), 8, C.c_void_p(host.ctypes.data), None) == -1
    assert L.md_velocity_sums_noalloc(None, 8, C.c_void_p(out.data_ptr()), None) == -1
    # the largest size it accepts, on an explicit stream
    big = torch.ones((md.NOALLOC_MAX_ATOMS, 3), dtype=torch.float64, device="cuda")
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        md.velocity_sums_noalloc(big, out=out)
    st.synchronize()
    n = float(md.NOALLOC_MAX_ATOMS)
    assert out.cpu().numpy().tolist() == [1.5 * n, n, n, n, float(np.sqrt(3.0))]
