"""mm_avg_m_noalloc (include/mm.h): the mean of m for callers that cannot allocate device memory, its scratch in a
file-scope device array. Checked against the existing path (mm_get_avg_m on a handle holding the same field) on two
calls in a row - the second on a different field, so stale partials or a stale ticket would show. Collected last
on purpose (file name): the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from synth import config_c1, random_unit_vectors

# both paths add the same fp32 values in fp64, in different orders: |sum| <= N, rounding <= N * 2^-53 per addition chain
AVG_TOL = 1e-12


@pytest.fixture(scope="module")
def mm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1406_7635_b200 import build
    build.build()
    import paper_1406_7635_b200 as mm
    return mm


def test_avg_m_noalloc_matches_mm_get_avg_m_on_two_calls_in_a_row(mm):
    import torch
    torch.cuda.set_device(0)
    grid = (200, 150, 3)                       # 90 000 cells: eleven 8192-cell chunks, the last one ragged
    n = grid[0] * grid[1] * grid[2]
    cfg = config_c1(grid=grid)
    sim = mm.from_config(cfg)
    out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.Stream()
    free_before = torch.cuda.mem_get_info()[0]
    for call, seed in enumerate((11, 12)):
        m0 = random_unit_vectors(seed, n).reshape(3, grid[2], grid[1], grid[0]).astype(np.float32)
        m0[0] += 0.25 * (call + 1)             # a mean well away from zero, different for the two calls
        sim.set_m(m0)                          # (normalises: the field both paths see is the handle's m)
        want = sim.avg_m()                     # existing path: k_sum3 with the handle's own scratch buffers
        m_dev = torch.from_numpy(sim.get_m()).cuda().contiguous()
        torch.cuda.synchronize()
        mm.avg_m_noalloc(m_dev, out, stream=stream.cuda_stream)
        stream.synchronize()
        got = out.cpu().numpy()
        assert np.all(np.isfinite(got))
        assert np.abs(got - want).max() <= AVG_TOL, (call, got, want)
        # and against a plain fp64 mean of the same floats
        assert np.abs(got - m_dev.cpu().numpy().astype(np.float64).reshape(3, -1).mean(axis=1)).max() <= AVG_TOL
        if call == 0:
            first = got.copy()
    assert np.abs(first - got).max() > 1e-3    # the second call did not just return the first call's result
    # same field again: same bits (fixed summation order), and the call itself took no device memory
    mm.avg_m_noalloc(m_dev, out, stream=stream.cuda_stream)
    stream.synchronize()
    assert np.array_equal(out.cpu().numpy(), got)
    assert torch.cuda.mem_get_info()[0] >= free_before - (8 << 20)      # (torch's own cache may have grown a little)


def test_avg_m_noalloc_rejects_what_it_cannot_do(mm):
    import torch
    lib = mm.lib()
    m = torch.zeros(3 * 64, dtype=torch.float32, device="cuda")
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    err = C.create_string_buffer(256)
    too_many = mm.MM_NOALLOC_MAX_CELLS + 1
    assert lib.mm_avg_m_noalloc(C.c_void_p(m.data_ptr()), too_many, C.c_void_p(out.data_ptr()), None, err, 256) == mm.MM_EINVAL
    assert b"MM_NOALLOC_MAX_CELLS" in err.value
    assert lib.mm_avg_m_noalloc(None, 64, C.c_void_p(out.data_ptr()), None, err, 256) == mm.MM_EINVAL
    assert lib.mm_avg_m_noalloc(C.c_void_p(m.data_ptr()), 0, C.c_void_p(out.data_ptr()), None, None, 0) == mm.MM_EINVAL
    host = np.zeros(3 * 64, dtype=np.float32)
    assert lib.mm_avg_m_noalloc(C.c_void_p(host.ctypes.data), 64, C.c_void_p(out.data_ptr()), None, err, 256) == mm.MM_EINVAL
    assert b"device memory" in err.value
    # a rejected call leaves the entry point usable
    m.fill_(0.5)
    mm.avg_m_noalloc(m, out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), np.full(3, 0.5))
