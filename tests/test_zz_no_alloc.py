"""cav_overlaps_noalloc (-m gpu): the entry point that allocates nothing (include/cavmag.h) against the existing,
handle-based path (cav_create + cav_get_dmdt + cav_get_overlaps) on the same device state, at the tolerances
tests/test_gpu_parity.py::test_rhs_matches_oracle uses for S (1e-14 in fp64, 2e-6 in fp32).

Collected last on purpose (the name sorts after every other test file): the suite runs with pytest -x, so a failure
here cannot hide another test.  Nothing here depends on what ran before: the scratch array is shared by every call in
the process and keeps the last call's contents, which is exactly what the back-to-back calls below exercise."""
import numpy as np
import pytest

from test_gpu_parity import small_problem

pytestmark = pytest.mark.gpu

S_TOL = {"f64": 1e-14, "f32": 2e-6}


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2603_03706_b200 import api as a      # raises if libcavmag.so is missing: no fallback
    return a


def existing_path(api, w, prec):
    """S_n and the device state m (as the library holds it after cav_set_m) from the handle-based path."""
    with api.Sim(w, precision=prec) as sim:
        dm = np.empty(sim.shape_m, dtype=sim.np_dtype)
        api.cav_get_dmdt(sim.h, dm)                              # one evaluation of the right-hand side
        S = api.cav_get_overlaps(sim.h, sim.N)
        m = sim.get_m()
    return np.asarray(S, dtype=np.complex128).reshape(-1), m       # (the binding returns complex numbers)


def no_alloc(api, torch, w, m, prec):
    dt = torch.float32 if prec == "f32" else torch.float64
    md = torch.as_tensor(np.ascontiguousarray(m), dtype=dt, device="cuda")
    ud = torch.as_tensor(np.ascontiguousarray(w.u), dtype=dt, device="cuda")
    N = ud.shape[0]
    out = torch.full((N, 2), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    return md, ud, out, stream


def as_complex(S):
    """[N][2] doubles (Re, Im), as cav_overlaps_noalloc writes them -> complex numbers"""
    S = np.asarray(S, dtype=np.float64).reshape(-1, 2)
    return S[:, 0] + 1j * S[:, 1]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("shape,N,n_sub", [
    ((72, 19, 5), 3, 1),        # one block, ragged
    ((68, 17, 6), 1, 2),        # antiferromagnet: m_c is the mean over the sublattices
    ((250, 33, 7), 8, 1),       # 57 750 cells: eight blocks, the last one ragged
    ((256, 64, 8), 8, 1),       # 131 072 cells: sixteen full blocks
    ((1, 1, 1), 1, 1),          # a single cell
])
def test_two_calls_in_a_row_match_the_existing_path(api, prec, shape, N, n_sub):
    import torch
    w = small_problem(*shape, N, n_sub)
    S_ref, m = existing_path(api, w, prec)
    md, ud, out, stream = no_alloc(api, torch, w, m, prec)
    grid = (w.nx, w.ny, w.nz)
    got = []
    for _ in range(2):                                           # the second call finds the first one's partials in the scratch
        out.fill_(float("nan"))
        api.cav_overlaps_noalloc(md, ud, out, grid, n_sub=n_sub, cuda_stream=stream)
        torch.cuda.synchronize()
        got.append(out.cpu().numpy().copy())
    assert np.array_equal(got[0], got[1])                        # fixed summation order: bitwise reproducible
    ref = S_ref
    assert np.abs(as_complex(got[0]) - ref).max() <= S_TOL[prec]
    # and against the definition (Eq. 18) on the same device state
    mc = np.asarray(m, dtype=np.float64).mean(axis=0)
    u = ud.cpu().numpy().astype(np.float64)
    S_def = np.array([(u[n] * (mc[0] - 1j * mc[1])).mean() for n in range(N)])
    assert np.abs(as_complex(got[0]) - S_def).max() <= S_TOL[prec]


def test_back_to_back_calls_on_different_problems(api):
    """A large call followed by a small one with fewer modes (stale partials of the first beyond the second's range),
    then the large one again: each equals the existing path's result for its own inputs."""
    import torch
    cases = [((256, 64, 8), 8, 1), ((20, 7, 6), 1, 2), ((256, 64, 8), 8, 1)]
    prepared = []
    for shape, N, n_sub in cases:
        w = small_problem(*shape, N, n_sub)
        S_ref, m = existing_path(api, w, "f64")
        prepared.append((w, n_sub, S_ref) + no_alloc(api, torch, w, m, "f64"))
    for w, n_sub, ref, md, ud, out, stream in prepared:          # enqueued back to back on one stream, one sync at the end
        api.cav_overlaps_noalloc(md, ud, out, (w.nx, w.ny, w.nz), n_sub=n_sub, cuda_stream=stream)
    torch.cuda.synchronize()
    for w, n_sub, ref, md, ud, out, stream in prepared:
        assert np.abs(as_complex(out.cpu().numpy()) - ref).max() <= S_TOL["f64"]


def test_it_allocates_nothing(api):
    import torch
    w = small_problem(250, 33, 7, 8, 1)
    md, ud, out, stream = no_alloc(api, torch, w, w.m0, "f32")
    grid = (w.nx, w.ny, w.nz)
    for _ in range(2):                                           # (the first call loads the module and finds the scratch array)
        api.cav_overlaps_noalloc(md, ud, out, grid, cuda_stream=stream)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(5):
        api.cav_overlaps_noalloc(md, ud, out, grid, cuda_stream=stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0


def test_limits_are_refused_with_a_reason(api):
    lib = api._lib
    one = 0x1000                                                 # never dereferenced: the sizes are checked first
    st = lib.cav_overlaps_noalloc(one, one, api.CAV_F32, 4096, 4096, 2, 1, 1, one, None)     # 2^25 cells
    assert st == api.CAV_E_UNSUPPORTED
    msg = api.cav_noalloc_last_error()
    assert "33554432 cells exceed the maximum of 16777216" in msg
    st = lib.cav_overlaps_noalloc(one, one, api.CAV_F32, 8, 8, 8, 1, 33, one, None)
    assert st == api.CAV_E_UNSUPPORTED and "33 modes exceed the maximum of 32" in api.cav_noalloc_last_error()
    assert lib.cav_overlaps_noalloc(one, one, 7, 8, 8, 8, 1, 1, one, None) == api.CAV_E_ARG
    assert lib.cav_overlaps_noalloc(None, one, api.CAV_F32, 8, 8, 8, 1, 1, one, None) == api.CAV_E_ARG
    assert lib.cav_overlaps_noalloc(one, one, api.CAV_F32, 8, 8, 8, 3, 1, one, None) == api.CAV_E_ARG
    # the largest size that is accepted: 2^24 cells, on real buffers
    import torch
    nx, ny, nz = 512, 512, 64
    m = torch.zeros((1, 3, nz, ny, nx), dtype=torch.float32, device="cuda")
    m[0, 0] = 0.6
    m[0, 1] = -0.8
    u = torch.ones((1, nz, ny, nx), dtype=torch.float32, device="cuda")
    out = torch.zeros((1, 2), dtype=torch.float64, device="cuda")
    api.cav_overlaps_noalloc(m, u, out, (nx, ny, nz), cuda_stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    S = out.cpu().numpy()[0]
    assert abs(S[0] - np.float32(0.6)) < 1e-12 and abs(S[1] - np.float32(0.8)) < 1e-12      # S = <m_x> - i <m_y>
    assert api.cav_noalloc_last_error() == ""
