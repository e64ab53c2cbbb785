"""Host logic of bench.py that needs no GPU: the algorithmic byte counts of SURVEY.md 8(d), the workload table with the
weak-scaling `zcopies`, and the slab-wise upload of a seeded state."""
import importlib.util
import os

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bench():
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_bytes_per_point_follow_the_survey(bench):
    """read w 40 + write w' 40 + read R_prev 40 (stages 1, 2) + write R 40 (stages 0, 1); +16 per stage with the lazy body
    force; +41 per stage with the sensor pass: 400 / 448 / 523 B per point per RK3 step."""
    assert bench.bytes_per_point_by_stage(dict(forcing=0, weno_enable=0)) == [120, 160, 120]
    assert sum(bench.bytes_per_point_by_stage(dict(forcing=0, weno_enable=0))) == 400
    assert bench.bytes_per_point_by_stage(dict(forcing=1, weno_enable=0)) == [136, 176, 136]
    assert sum(bench.bytes_per_point_by_stage(dict(forcing=1, weno_enable=0))) == 448
    assert sum(bench.bytes_per_point_by_stage(dict(forcing=0, weno_enable=1))) == 523


def test_workload_table_and_weak_scaling_copies(bench):
    wl = bench.make_workload(5)
    assert (wl.grid["nx"], wl.grid["ny"], wl.grid["nz"]) == (1024, 512, 512) and wl.params["forcing"] == 1
    w4 = bench.make_workload(5, zcopies=4)
    assert w4.grid["nz"] == 2048 and w4.grid["len"][2] == pytest.approx(4 * wl.grid["len"][2])
    assert w4.z[1] - w4.z[0] == pytest.approx(wl.z[1] - wl.z[0])               # same spacing: one box per GPU
    s4 = bench.make_workload(4, zcopies=2)
    assert s4.grid["nz"] == 256 and s4.params["weno_enable"] == 1
    with pytest.raises(SystemExit):
        bench.make_workload(2, zcopies=2)
    with pytest.raises(SystemExit):
        bench.make_workload(9)


def test_upload_state_in_slabs_equals_the_seeded_state(bench):
    import workloads as W
    wl = W.config3_channel(16, 8, 20)
    full = wl.state()
    up = bench.upload_state(torch, wl, "cpu", planes=6)
    assert np.array_equal(up.numpy(), full)
    part = bench.upload_state(torch, wl, "cpu", planes=4, k0=5, k1=17)
    assert np.array_equal(part.numpy(), full[:, 5:17])
