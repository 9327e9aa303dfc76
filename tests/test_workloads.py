"""The seeded input generators: deterministic, right shapes/dtypes/statistics, no method arithmetic."""
import numpy as np

from paper_1107_5578_b200 import workloads as W


def test_configs_match_baseline_json():
    c = W.CONFIGS
    assert (c["c1"].N, c["c1"].lam, c["c1"].pitch, c["c1"].zs) == (256, 633e-9, 10e-6, (0.05,))
    assert (c["c2"].N, c["c2"].lam, c["c2"].pitch, c["c2"].zs) == (1024, 532e-9, 8e-6, (0.2,))
    assert (c["c3"].N, c["c3"].lam, c["c3"].pitch, c["c3"].zs) == (4096, 633e-9, 4e-6, (0.01, 0.1, 0.5))
    assert c["c4"].N == 2048 and len(c["c4"].zs) == 64 and abs(c["c4"].zs[63] - 0.064) < 1e-15
    assert (c["c5"].N, c["c5"].pitch, c["c5"].zs, c["c5"].iters) == (8192, 3.74e-6, (0.3,), 20)


def test_fields_are_deterministic_and_shaped():
    for name in ("c1", "c2", "c3", "c4"):
        cfg = W.CONFIGS[name].scaled(64)
        a = W.make_field(cfg); b = W.make_field(cfg)
        assert a.dtype == np.complex64 and a.shape == (64, 64) and np.array_equal(a, b)
    a = W.make_field(W.CONFIGS["c2"].scaled(256))
    assert set(np.unique(a)) == {0, 1} and 0.03 < a.real.mean() < 0.07
    a = W.make_field(W.CONFIGS["c4"].scaled(64))
    assert np.allclose(np.abs(a), 1, atol=1e-6)
    a = W.make_field(W.CONFIGS["c3"].scaled(256))
    assert abs(a.real.std() - 1) < 0.02 and abs(a.imag.std() - 1) < 0.02
    a = W.make_field(W.CONFIGS["c1"].scaled(256))
    assert np.abs(a).max() < 1 and abs(np.abs(a).mean() - 0.5) < 0.02


def test_gs_inputs():
    cfg = W.CONFIGS["c5"].scaled(128)
    s, d, p = W.gs_inputs_c5(cfg)
    assert s.dtype == d.dtype == p.dtype == np.float32
    assert np.all(s == 1) and abs(np.sum(d.astype(float) ** 2) / np.sum(s.astype(float) ** 2) - 1) < 1e-5
    assert 0 <= p.min() and p.max() < 2 * np.pi + 1e-6
    # 9x9 blur: neighbouring samples are strongly correlated
    assert np.corrcoef(d[:, :-1].ravel(), d[:, 1:].ravel())[0, 1] > 0.8
