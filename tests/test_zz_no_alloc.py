"""nf_max_speed_static, the entry point that allocates nothing (include/nf.h): its output against the existing
nf_max_speed path on two calls in a row -- the second on a field with a SMALLER maximum and a different size, so that
partial maxima left in the shared static scratch by the first call would show.  The maximum is exact in both paths:
the comparison is bit-for-bit (the tolerance every max-speed test here uses).  Collected last on purpose (file name)."""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


@pytest.fixture(scope="module")
def api():
    from paper_2405_14903_b200 import api as a
    a.load_library()
    return a


def _fields(torch, nx, ny, nz, seed, scale):
    rng = np.random.default_rng(seed)
    shapes = ((nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx))
    return [torch.from_numpy((scale * rng.standard_normal(s)).astype(np.float32)).cuda() for s in shapes]


def test_static_max_speed_matches_the_handle_path_twice_in_a_row(torch, api):
    out = torch.full((1,), -1.0, dtype=torch.float32, device="cuda")
    # first call: 72 x 40 x 52 (10 partial maxima per component, ragged last segment), large values;
    # second call: a smaller grid with values 100 times smaller (stale partials of call one must not be read)
    for (nx, ny, nz), seed, scale in (((72, 40, 52), 5, 3.0), ((40, 36, 28), 6, 0.03)):
        U = _fields(torch, nx, ny, nz, seed, scale)
        g = api.Grid(nx, ny, nz, 1.0 / nx)
        ref = g.max_speed(*U)                      # the existing path (handle, scratch word in the handle)
        g.close()
        api.max_speed_static(U[0], U[1], U[2], out)
        got = float(out.cpu()[0])
        assert got == ref, (got, ref)
        assert got == max(float(a.abs().max()) for a in U)


def test_static_max_speed_repeats_and_propagates_nan(torch, api):
    U = _fields(torch, 64, 64, 64, 7, 1.0)
    out = torch.zeros(1, dtype=torch.float32, device="cuda")
    first = float(api.max_speed_static(*U, out).cpu()[0])
    second = float(api.max_speed_static(*U, out).cpu()[0])
    assert first == second == max(float(a.abs().max()) for a in U)
    U[1][3, 4, 5] = float("nan")
    assert np.isnan(float(api.max_speed_static(*U, out).cpu()[0]))


def test_static_max_speed_rejects_sizes_beyond_its_scratch(torch, api):
    lib = api.load_library()
    dummy = torch.zeros(8, dtype=torch.float32, device="cuda")
    p = ctypes.c_void_p(dummy.data_ptr())
    # 512^3: 3 x 8208 partial maxima > 16384 -- rejected before anything is launched or read
    rc = lib.nf_max_speed_static(p, p, p, 512, 512, 512, None, p)
    assert rc == -1
    msg = lib.nf_static_last_error().decode()
    assert "16384" in msg and "512" in msg
    assert lib.nf_max_speed_static(None, p, p, 8, 8, 8, None, p) == -1
    assert lib.nf_max_speed_static(p, p, p, 0, 8, 8, None, p) == -1
    torch.cuda.synchronize()
