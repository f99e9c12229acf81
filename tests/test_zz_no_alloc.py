"""mpr_sample_energy_static (include/mpr.h; csrc/mpr_static.cu): the entry point that takes no workspace and allocates
nothing -- its intermediates live in a file-scope device array of the library.  Checked against the existing path
(mpr_create + mpr_sample_energy + mpr_get_info, which keeps the same intermediates in the caller's workspace) within
the tolerance the set-up parity tests use (1e-12 relative on e_s, exact on counts and range), on calls in a row that
share the array: the second call must not see anything of the first.  Collected last on purpose (the suite runs with
pytest -x); passes alone in a fresh process and after the other tests."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mpr():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1910_08448_b200 import build, mpr as m
    build.build()
    m.lib()
    return m


@pytest.fixture(scope="module")
def inputs():
    from paper_1910_08448_b200 import inputs as i
    return i


def existing_path(mpr, values, mask):
    """(e_s, pairs, z_min, z_max) by the context path, workspace and all."""
    g = mpr.Mpr(values, mask)
    e_s, n_pairs = g.sample_energy()
    info = g.info()
    g.close()
    return e_s, n_pairs, info["z_min"], info["z_max"]


def check(mpr, out, values, mask):
    e_s, n_pairs, z_min, z_max = existing_path(mpr, values, mask)
    got = out.cpu().numpy()
    assert got[1] == n_pairs
    assert got[2] == z_min and got[3] == z_max
    assert abs(got[0] - e_s) <= 1e-12 * abs(e_s), (got[0], e_s)
    assert got[4] == int((mask == 0).sum()) and got[5] == 0.0


def test_two_calls_in_a_row_match_the_workspace_path(mpr, inputs):
    import torch
    assert mpr.lib().mpr_static_setup() == mpr.MPR_OK
    dev = torch.device("cuda:0")
    out = torch.full((6,), -1.0, dtype=torch.float64, device=dev)
    # a large problem first (all 1024 partial slots written), then a small rectangular one (3 blocks): the second call
    # reads only what it wrote although the array still holds the first call's partials
    big = inputs.make_problem(700, 12.0, 31, 0.6)
    small = inputs.make_rect_problem(23, 31, 5.0, 32, 0.4)
    for n, (values, mask, _) in enumerate((big, small, big)):
        dv, dm = torch.from_numpy(values).to(dev), torch.from_numpy(mask).to(dev)
        torch.cuda.synchronize(dev)
        free_before = torch.cuda.mem_get_info(dev)[0]
        mpr.sample_energy_static(dv, dm, out)
        torch.cuda.synchronize(dev)
        if n > 0:       # (the first call may make the driver load the four kernels: code, not data)
            assert torch.cuda.mem_get_info(dev)[0] == free_before        # the call took no device memory
        check(mpr, out, values, mask)


def test_back_to_back_without_a_sync_in_between(mpr, inputs):
    """Two calls enqueued on one stream with no synchronisation between them (the order the stream gives is the only
    thing that keeps them apart), each into its own output."""
    import torch
    dev = torch.device("cuda:0")
    a = inputs.make_problem(300, 8.0, 41, 0.9)
    b = inputs.make_problem(180, 6.0, 42, 0.33, True)
    ta = [torch.from_numpy(x).to(dev) for x in a[:2]]
    tb = [torch.from_numpy(x).to(dev) for x in b[:2]]
    oa = torch.zeros(6, dtype=torch.float64, device=dev)
    ob = torch.zeros(6, dtype=torch.float64, device=dev)
    torch.cuda.synchronize(dev)
    mpr.sample_energy_static(ta[0], ta[1], oa)
    mpr.sample_energy_static(tb[0], tb[1], ob)
    torch.cuda.synchronize(dev)
    check(mpr, oa, a[0], a[1])
    check(mpr, ob, b[0], b[1])


def test_undefined_cases_and_limits(mpr):
    import torch
    dev = torch.device("cuda:0")
    out = torch.zeros(6, dtype=torch.float64, device=dev)
    L = 16
    rng = np.random.default_rng(3)
    z = torch.from_numpy(rng.normal(50, 10, (L, L))).to(dev)
    # no measured pair: every other site measured on a checkerboard
    yy, xx = np.mgrid[0:L, 0:L]
    cb = torch.from_numpy(((xx + yy) & 1).astype(np.uint8)).to(dev)
    got = mpr.sample_energy_static(z, cb, out).cpu().numpy()
    assert math.isnan(got[0]) and got[1] == 0 and got[4] == L * L // 2
    # constant sample: degenerate range
    got = mpr.sample_energy_static(torch.full((L, L), 3.0, dtype=torch.float64, device=dev),
                                   torch.zeros((L, L), dtype=torch.uint8, device=dev), out).cpu().numpy()
    assert math.isnan(got[0]) and got[2] == got[3] == 3.0
    # beyond the stated maximum: rejected before anything is launched or read, with a message
    assert mpr.static_max_sites() == 1 << 28
    with pytest.raises(mpr.MprError) as ei:
        mpr.sample_energy_static(z, cb, out, shape=(16384, 16385))
    assert ei.value.code == mpr.ERR_INVALID_ARG and "exceed" in str(ei.value)
    with pytest.raises(mpr.MprError):
        mpr.sample_energy_static(z, cb, out, q=0.75)
    # and a valid call afterwards still works
    m0 = torch.zeros((L, L), dtype=torch.uint8, device=dev)
    got = mpr.sample_energy_static(z, m0, out).cpu().numpy()
    assert got[1] == 2 * L * (L - 1) and not math.isnan(got[0])


def test_captured_in_a_cuda_graph(mpr, inputs):
    """The reason the entry point exists: it can be recorded into a CUDA graph (no allocation, no synchronisation, no
    host read-back inside the call) and replayed on new data in the same buffers."""
    import torch
    dev = torch.device("cuda:0")
    assert mpr.lib().mpr_static_setup() == mpr.MPR_OK         # the symbol's address is taken before the capture
    a = inputs.make_problem(200, 8.0, 61, 0.5)
    b = inputs.make_problem(200, 8.0, 62, 0.7)
    dv, dm = torch.from_numpy(a[0]).to(dev), torch.from_numpy(a[1]).to(dev)
    out = torch.zeros(6, dtype=torch.float64, device=dev)
    side = torch.cuda.Stream(device=dev)
    side.wait_stream(torch.cuda.current_stream(dev))
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        mpr.sample_energy_static(dv, dm, out, stream=side)    # warm-up outside the capture (loads the kernels)
        side.synchronize()
        with torch.cuda.graph(graph, stream=side):
            mpr.sample_energy_static(dv, dm, out, stream=side)
    torch.cuda.current_stream(dev).wait_stream(side)
    out.zero_()
    graph.replay()
    torch.cuda.synchronize(dev)
    check(mpr, out, a[0], a[1])
    dv.copy_(torch.from_numpy(b[0]))                           # new data in the same buffers, same graph
    dm.copy_(torch.from_numpy(b[1]))
    graph.replay()
    torch.cuda.synchronize(dev)
    check(mpr, out, b[0], b[1])
