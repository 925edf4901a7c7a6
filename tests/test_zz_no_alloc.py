"""mfc_cfl_dt_static — the CFL time step for callers that must not allocate — against the existing path.

Who needs it: a solver that runs inside an application whose memory pool already owns the GPU's memory (a further
cudaMalloc fails or fragments the pool), or a time-step loop in which an allocation would stall the whole device.  Such
a caller cannot create an mfc_grid (mfc_init_grid allocates), so the entry point takes the grid description directly
and keeps its reduction scratch in an array built into the library (129 KiB per GPU, at most 2^25 cells).

The reference here is the path that already exists and is itself compared with the CPU reference bit for bit in
test_gpu_parity.py::test_cfl_dt_bit_exact: Grid.cfl_dt (mfc_init_grid + mfc_cfl_dt).  Both evaluate the same IEEE
operations per cell and a maximum, so the bar is the one that test uses: equality of the bits.

Every test makes (at least) two calls in a row without synchronising in between: the array is shared by all calls and
keeps the previous call's contents, so the second call is the one that shows whether it starts clean.  The file is
named to be collected last (pytest -x stops at the first failure; a failure here must not hide other tests) and does
not depend on what ran before it: the device address of the array is looked up by whichever call comes first."""
import ctypes as C

import pytest

import mfc_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    return t


@pytest.fixture(scope="module")
def mfc():
    import paper_2503_07953_b200 as m
    m.lib()
    return m


def static_dt(torch, mfc, case, qd, cfl):
    """(dt tensor, flag tensor) of one asynchronous call; nothing is synchronised here"""
    dt = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    flag = torch.full((1,), -7, dtype=torch.int32, device="cuda")
    mfc.cfl_dt_static(case.ndim, case.n, case.dx, case.gamma, case.pi_inf, qd, cfl, dt, flag)
    return dt, flag


# sizes: one block only, a ragged last block, several hundred blocks; 1-3 fluids, 1-3 dimensions
@pytest.mark.parametrize("index,n", [(1, None), (2, None), (3, 200), (4, 50), (5, 44), (4, 97)])
def test_two_calls_in_a_row_equal_the_handle_path_bit_for_bit(torch, mfc, index, n):
    case = W.config(index, n=n)
    qa = torch.from_numpy(W.initial_state(case)).cuda()
    qb = torch.from_numpy(W.random_admissible_state(case, seed=11)).cuda()
    g = mfc.Grid.from_case(case)
    want_a, want_b = g.cfl_dt(qa, case.cfl), g.cfl_dt(qb, 0.5 * case.cfl)
    assert want_a != want_b
    got_a = static_dt(torch, mfc, case, qa, case.cfl)           # first call
    got_b = static_dt(torch, mfc, case, qb, 0.5 * case.cfl)     # second call, enqueued right behind it
    got_a2 = static_dt(torch, mfc, case, qa, case.cfl)          # and the first state again
    torch.cuda.synchronize()
    assert got_a[0].item() == want_a and got_a[1].item() == 0
    assert got_b[0].item() == want_b and got_b[1].item() == 0
    assert got_a2[0].item() == want_a and got_a2[1].item() == 0


def test_flag_of_a_nonphysical_state_does_not_leak_into_the_next_call(torch, mfc):
    case = W.config(3, n=160)
    good = W.random_admissible_state(case, seed=3)
    bad = good.copy()
    bad[0, 0, 17, 33] = -5000.0  # mixture density below zero in one cell
    gd, bd = torch.from_numpy(good).cuda(), torch.from_numpy(bad).cuda()
    want = mfc.Grid.from_case(case).cfl_dt(gd, case.cfl)
    r1 = static_dt(torch, mfc, case, bd, case.cfl)
    r2 = static_dt(torch, mfc, case, gd, case.cfl)
    r3 = static_dt(torch, mfc, case, gd, case.cfl)
    torch.cuda.synchronize()
    assert r1[1].item() == 1
    assert r2[1].item() == 0 and r2[0].item() == want
    assert r3[1].item() == 0 and r3[0].item() == want
    # the flag output is optional
    dt = torch.zeros(1, dtype=torch.float64, device="cuda")
    mfc.cfl_dt_static(case.ndim, case.n, case.dx, case.gamma, case.pi_inf, gd, case.cfl, dt, None)
    torch.cuda.synchronize()
    assert dt.item() == want


def test_largest_grid_the_array_holds_and_refusal_beyond_it(torch, mfc):
    n = mfc.STATIC_MAX_CELLS  # 2^25 cells in one dimension, one fluid: every one of the 16384 partial results is used
    gamma, pi_inf = (1.4,), (0.0,)
    dx = (1.0 / n, 1.0, 1.0)
    gen = torch.Generator(device="cuda").manual_seed(5)
    rho = 1.0 + torch.rand(n, dtype=torch.float64, device="cuda", generator=gen)
    u = 200.0 * (torch.rand(n, dtype=torch.float64, device="cuda", generator=gen) - 0.5)
    p = 1.0e5 * (1.0 + torch.rand(n, dtype=torch.float64, device="cuda", generator=gen))
    u[n - 1] = 4000.0  # the maximum sits in the very last cell of the very last block
    q = torch.stack([rho, rho * u, p / 0.4 + 0.5 * rho * u * u, torch.ones_like(rho)]).contiguous()
    del rho, u, p
    g = mfc.Grid(1, (n, 1, 1), dx, gamma, pi_inf, (W.BC_EXTRAP,) * 3, (W.BC_EXTRAP,) * 3)
    want = g.cfl_dt(q, 0.4)
    g.close()
    outs = []
    for _ in range(2):
        dt = torch.zeros(1, dtype=torch.float64, device="cuda")
        flag = torch.full((1,), -1, dtype=torch.int32, device="cuda")
        mfc.cfl_dt_static(1, (n, 1, 1), dx, gamma, pi_inf, q, 0.4, dt, flag)
        outs.append((dt, flag))
    torch.cuda.synchronize()
    for dt, flag in outs:
        assert dt.item() == want and flag.item() == 0
    # one cell more: refused before anything is launched (q is not touched, so a short array will do), outputs untouched
    p_ = mfc.MfcParams()
    p_.ndim, p_.nfluids, p_.device = 2, 1, 0
    ga, pa = (C.c_double * 1)(1.4), (C.c_double * 1)(0.0)
    p_.gamma, p_.pi_inf = C.cast(ga, C.POINTER(C.c_double)), C.cast(pa, C.POINTER(C.c_double))
    for d, (nd, h) in enumerate([(4097, 1e-3), (8192, 1e-3), (1, 1.0)]):
        p_.n[d], p_.dx[d] = nd, h
    p_.stream = torch.cuda.current_stream().cuda_stream
    dt = torch.full((1,), -3.0, dtype=torch.float64, device="cuda")
    st = mfc.lib().mfc_cfl_dt_static(C.byref(p_), q.data_ptr(), 0.4, dt.data_ptr(), None)
    assert st == mfc.MFC_ERR_ARG
    text = mfc.lib().mfc_last_error().decode()
    assert "too large" in text and str(mfc.STATIC_MAX_CELLS) in text
    torch.cuda.synchronize()
    assert dt.item() == -3.0


def test_argument_errors_are_reported_not_launched(torch, mfc):
    case = W.config(1)
    q = torch.from_numpy(W.initial_state(case)).cuda()
    dt = torch.zeros(1, dtype=torch.float64, device="cuda")
    with pytest.raises(mfc.MfcError) as e:
        mfc.cfl_dt_static(case.ndim, case.n, (0.0, 1.0, 1.0), case.gamma, case.pi_inf, q, 0.5, dt)
    assert e.value.status == mfc.MFC_ERR_ARG
    with pytest.raises(mfc.MfcError) as e:
        mfc.cfl_dt_static(case.ndim, case.n, case.dx, (1.0,) * case.nfluids, case.pi_inf, q, 0.5, dt)
    assert e.value.status == mfc.MFC_ERR_ARG
    with pytest.raises(mfc.MfcError) as e:
        mfc.cfl_dt_static(case.ndim, case.n, case.dx, case.gamma, case.pi_inf, q, 0.5, dt, device=99, stream=0)
    assert e.value.status == mfc.MFC_ERR_ARG
