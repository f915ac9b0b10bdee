"""dg_torque_static (include/dg.h): the entry point that allocates nothing -- its reduction scratch is a static
__device__ array inside the library -- against the existing path, dg_torque (scratch in the caller's workspace), and
against the CPU oracle, at the tolerance of test_parity_gpu.test_torque_parity.  Collected last on purpose (the name):
`pytest -x` must not lose the parity tests to a failure here."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from paper_1805_01443_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-12


@pytest.fixture(scope="module")
def lib():
    from paper_1805_01443_b200 import dg
    from paper_1805_01443_b200.build import build
    build()
    dg.load_library()
    return dg


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _scale(p, U):
    """sum_n |M_n|: what the rounding of the sum is relative to (the torque itself cancels)."""
    return np.abs(U[..., 0, 0, 0]).sum() * (p["x1"] - p["x0"]) / p["nx"] * (p["y1"] - p["y0"]) / p["ny"]


# several 32 x 32 blocks with ragged tails in both directions; one block; less than one block
GRIDS = [(70, 45, 3, 0, 1), (64, 40, 5, 1, 2), (33, 7, 4, 1, 2), (32, 32, 2, 0, 1), (5, 3, 1, 0, 1)]


@pytest.mark.parametrize("nx,ny,m,eos,bc", GRIDS)
def test_torque_static_matches_dg_torque_on_two_calls_in_a_row(lib, nx, ny, m, eos, bc):
    p, U = W.random_smooth(nx, ny, m, seed=21, eos=eos, bc=bc, gravity=True)
    Ud = dev(U)
    g = lib.DG(p)
    g.set_state(Ud)
    ref = oracle.RefDG(p)
    ref.set_state(U)
    out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
    tol = TOL * _scale(p, U)
    # two calls in a row into the same output and the same static scratch, at different times
    for t in (0.0, 1.7):
        lib.torque_static(p, Ud, t, out)
        got = out.cpu().numpy().copy()
        want = g.torque(t)
        assert abs(got[0] - want) < max(tol, TOL * abs(want)), (t, got[0], want)
        gr = ref.torque(t)
        assert abs(got[0] - gr) < max(tol, TOL * abs(gr)), (t, got[0], gr)
        ang = p["omega_planet"] * t + p["phase0"]
        xp, yp = p["r_planet"] * np.cos(ang), p["r_planet"] * np.sin(ang)
        assert abs(got[0] - (xp * got[2] - yp * got[1])) <= 1e-14 * (abs(xp * got[2]) + abs(yp * got[1]))
    # the same call again gives the same bits (fixed summation order, nothing left over in the scratch matters)
    again = torch.empty(3, dtype=torch.float64, device="cuda")
    lib.torque_static(p, Ud, 1.7, again)
    assert torch.equal(again, out)


def test_a_small_grid_after_a_large_one_sees_none_of_its_scratch(lib):
    """The array keeps the last call's contents: a call must read only the slots it wrote itself."""
    pb, Ub = W.random_smooth(300, 130, 2, seed=22, eos=0, bc=1, gravity=True)
    ps, Us = W.random_smooth(37, 9, 2, seed=23, eos=0, bc=1, gravity=True)
    out = torch.empty(3, dtype=torch.float64, device="cuda")
    gb = lib.DG(pb)
    gb.set_state(dev(Ub))
    lib.torque_static(pb, dev(Ub), 0.3, out)
    want = gb.torque(0.3)
    assert abs(out[0].item() - want) < max(TOL * _scale(pb, Ub), TOL * abs(want))
    gs = lib.DG(ps)
    gs.set_state(dev(Us))
    lib.torque_static(ps, dev(Us), 0.3, out)
    want = gs.torque(0.3)
    assert abs(out[0].item() - want) < max(TOL * _scale(ps, Us), TOL * abs(want))


def test_runs_on_the_callers_stream_and_allocates_nothing(lib):
    p, U = W.random_smooth(70, 45, 3, seed=24, eos=0, bc=1, gravity=True)
    Ud = dev(U)
    g = lib.DG(p)
    g.set_state(Ud)
    want = g.torque(0.9)
    out = torch.empty(3, dtype=torch.float64, device="cuda")
    lib.static_setup()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    lib.torque_static(p, Ud, 0.9, out, stream=s)    # (the first launch of a kernel loads its code)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        lib.torque_static(p, Ud, 0.9, out, stream=s)
    s.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                       # no device memory was taken by the calls
    assert abs(out[0].item() - want) < max(TOL * _scale(p, U), TOL * abs(want))


def test_sizes_beyond_the_static_scratch_are_rejected(lib):
    import ctypes as C
    L = lib.load_library()
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    U = torch.zeros(8, dtype=torch.float64, device="cuda")     # never read: the size check comes first
    p = W.make_params(nx=32 * 512, ny=32 * 129, order=1, x0=-1.0, x1=1.0, y0=-1.0, y1=1.0)   # 66 048 blocks > 65 536
    e = L.dg_torque_static(C.byref(lib.params_struct(p)), U.data_ptr(), 0.0, out.data_ptr(), None)
    assert e == -2                                             # DG_ENOSPC
    msg = L.dg_static_last_error().decode()
    assert "DG_STATIC_MAX_BLOCKS" in msg and "66048" in msg
    torch.cuda.synchronize()
    assert (out == 0).all()                                    # nothing was launched
    with pytest.raises(lib.DGError):
        lib.torque_static(p, U, 0.0, out)                      # the binding's own size check
