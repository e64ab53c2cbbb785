"""streams_max_speed_static (include/streams.h): the S10 maxima through the entry point that allocates nothing (its scratch
is a file-scope static device array of the library) against the existing path (streams_set_state + streams_diagnostics,
scratch in the caller's workspace).  Collected last on purpose (file name): the suite runs with pytest -x.

The two paths evaluate the same expression on the same state and a maximum is exact, so the tolerance is the tightest
one of the GPU tests (1e-12 relative, FMA contraction may differ between the two kernels); the existing path itself is
checked against the CPU oracle in test_gpu_parity.py.
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def env():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2004_02276_b200 import build
    build.build()
    from paper_2004_02276_b200 import binding
    binding.lib()
    return torch, binding


def existing_path(binding, torch, wl, w):
    c = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    c.set_state(w)
    ref = np.array(c.diagnostics().max_speed[:])
    c.close()
    return ref


def test_two_calls_in_a_row_equal_the_existing_path(env):
    """Call 1: 60 CTAs of a stretched channel; call 2, straight after it on another context: 3 CTAs of a small box with
    lower speeds (a stale partial or ticket of call 1 in the shared static array would show); call 3: call 1 again."""
    torch, binding = env
    big = W.config3_channel(96, 64, 80)                      # 491 520 nodes, ragged last CTA
    small = W.random_periodic(33, 17, 29, params=W.default_params(Rgas=1 / 1.4, mu_ref=5e-3), stretched_y=True)
    wb = torch.from_numpy(big.state()).cuda()
    ws = torch.from_numpy(0.5 * small.state()).cuda()
    ref_b = existing_path(binding, torch, big, wb)
    ref_s = existing_path(binding, torch, small, ws)
    assert np.all(ref_b > 0) and np.all(ref_s > 0) and not np.allclose(ref_b, ref_s)
    cb = binding.Streams(big.grid, big.x, big.y, big.z, big.params)         # no state set: the input is the argument
    cs = binding.Streams(small.grid, small.x, small.y, small.z, small.params)
    out = torch.full((3, 3), -1.0, dtype=torch.float64, device="cuda")
    cb.max_speed_static(wb, out[0])
    cb.stream.synchronize()                                  # calls that overlap on the GPU would race on the array
    free0 = torch.cuda.mem_get_info()[0]
    n0 = cs.launch_count()
    cs.max_speed_static(ws, out[1])
    cs.stream.synchronize()
    cb.max_speed_static(wb, out[2])
    cb.stream.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0             # nothing was allocated on the device
    assert cs.launch_count() == n0 + 1                       # one kernel
    got = out.cpu().numpy()
    for g, r in ((got[0], ref_b), (got[1], ref_s), (got[2], ref_b)):
        assert np.all(np.abs(g - r) <= TOL * np.abs(r)), (g, r)
    # back to back on ONE stream without a host synchronisation in between
    out.fill_(-1.0)
    torch.cuda.synchronize()
    for row in range(3):
        cb.max_speed_static(wb, out[row])
    cb.stream.synchronize()
    got = out.cpu().numpy()
    assert np.all(np.abs(got - ref_b) <= TOL * np.abs(ref_b)), (got, ref_b)
    cb.close()
    cs.close()


def test_sizes_beyond_the_static_array_are_rejected(env):
    torch, binding = env
    assert binding.Streams.STATIC_MAX_NODES == 8192 * 4096
    wl = W.random_periodic(520, 256, 256)                    # 34.1 M nodes > 33 554 432; the state is never generated
    c = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    w = torch.empty((5, 256, 256, 520), dtype=torch.float64, device="cuda")
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    with pytest.raises(binding.StreamsError) as ei:
        c.max_speed_static(w, out)
    assert ei.value.code == binding.STREAMS_EINVAL and "static scratch limit" in str(ei.value)
    assert float(out.abs().max()) == 0.0
    c.close()
