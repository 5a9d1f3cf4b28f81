"""The seeded input generator (paper_0809_3098_b200/workloads.py): holds no arithmetic of the method."""
import os

import numpy as np

from paper_0809_3098_b200 import workloads as W


def test_lcg_vectorised_equals_recurrence():
    for seed in (1, 80930981, 2 ** 63 + 12345):
        assert np.array_equal(W.lcg_uniform(seed, 1000), W.lcg_uniform_loop(seed, 1000))
    assert W.lcg_uniform(5, 0).size == 0


def test_lcg_first_draw_by_hand():
    s = (80930981 * 6364136223846793005 + 1442695040888963407) % 2 ** 64
    assert W.lcg_uniform(80930981, 1)[0] == (s >> 11) / 2.0 ** 53


def test_configs_follow_baseline_json():
    c = [W.config(k) for k in range(1, 6)]
    assert [x.N for x in c] == [32, 128, 512, 1024, 1024]
    assert [x.Re for x in c] == [100.0, 1000.0, 5000.0, 10000.0, 30000.0]
    assert c[0].dt == 0.0156                                    # literal (G13)
    for x in c[1:]:
        h = 1.0 / x.N
        assert x.dt == min(0.5 * h, 0.2 * h * h * x.Re) == 0.5 * h
    assert [x.sweeps_per_stage for x in c] == [20, 50, 100, 200, 200]
    assert [x.sor_omega for x in c] == [1.8, 1.95, 1.99, 1.995, 1.995]
    assert [x.steps for x in c] == [200, 2000, 5000, 1000, 1000]
    assert c[4].poisson_sweeps == 10000 and c[4].smooth_amp == 5.0 and c[4].noise == 1e-3


def test_initial_fields_shape_ring_and_range():
    wl = W.config(1)
    psi, w = W.initial_fields(wl)
    assert psi.shape == w.shape == (33, 33) and not psi.any()
    assert not w[0].any() and not w[-1].any() and not w[:, 0].any() and not w[:, -1].any()
    assert np.all(np.abs(w[1:-1, 1:-1]) <= 1e-6) and np.count_nonzero(w[1:-1, 1:-1]) > 900
    # row-major order of the draws: first interior point (j=1, i=1) takes the first draw
    assert w[1, 1] == 1e-6 * (2.0 * W.lcg_uniform(wl.seed, 1)[0] - 1.0)
    assert w[1, 2] == 1e-6 * (2.0 * W.lcg_uniform(wl.seed, 2)[1] - 1.0)


def test_config5_smooth_part():
    wl = W.config(5)
    w = W.initial_omega(64, 0.0, 1, smooth_amp=5.0)
    assert abs(w[16, 16] - 5.0) < 1e-12 and abs(w[48, 16] + 5.0) < 1e-12
    assert wl.smooth_amp == 5.0


def test_bench_ncu_traffic_constant_is_tied_to_the_kernel_sources(tmp_path, monkeypatch):
    # roofline.traffic is an ncu figure of ONE build: bench.py may report it only while the kernel sources are unchanged
    import bench
    assert set(bench.NCU_DRAM_BUILD) >= {"paper_0809_3098_b200/csrc/cavity_resident.cu"}
    assert bench.ncu_capture_is_current() in (True, False)      # a changed kernel is not an error: bench.py then prints traffic: null
    import hashlib
    data = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "README.md"), "rb").read()
    monkeypatch.setattr(bench, "NCU_DRAM_BUILD", {"README.md": hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()})
    assert bench.ncu_capture_is_current()                        # the id is git's blob id of the file's bytes
    monkeypatch.setattr(bench, "NCU_DRAM_BUILD", {"paper_0809_3098_b200/csrc/cavity_resident.cu": "0" * 40})
    assert not bench.ncu_capture_is_current()
