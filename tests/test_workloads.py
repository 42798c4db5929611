"""The seeded input generator: determinism, independence of generation order, and that the
achieved shapes match BASELINE.json configs (readings A15-A19).  CPU only."""
import numpy as np
import pytest

from paper_2004_04334_b200 import workloads as wl


def test_deterministic_and_order_independent():
    a = wl.make_event(1, 3)
    wl.make_event(3, 0)
    b = wl.make_event(1, 3)
    assert np.array_equal(a.words, b.words) and np.array_equal(a.adc, b.adc)
    c = wl.make_event(1, 4)
    assert not np.array_equal(a.words[:1000], c.words[:1000])
    assert not np.array_equal(wl.make_event(1, 3, seed=1).words[:1000], a.words[:1000])
    g1, g2 = wl.make_calib(1), wl.make_calib(1)
    assert np.array_equal(g1.gain, g2.gain) and np.array_equal(g1.pedestal, g2.pedestal)


@pytest.mark.parametrize("config,D,N,f,tol", [(0, 2000, 670, 0.01, 0.15), (1, 50000, 8000, 0.005, 0.06),
                                              (3, 200000, 30000, 0.005, 0.04)])
def test_shapes_match_configs(config, D, N, f, tol):
    evs = [wl.make_event(config, e) for e in range(4)]
    d = np.mean([e.stats["n_digis"] for e in evs])
    n = np.mean([e.stats["n_seeded_clusters"] for e in evs])
    assert abs(d - D) / D < tol and abs(n - N) / N < tol
    for e in evs:
        assert abs(e.stats["n_errors"] / e.stats["n_words"] - f) < 0.1 * f + 1e-4
        err = (e.words >> 31) == 1
        assert int(err.sum()) == e.stats["n_errors"] and np.all(e.adc[err] == 0)
        v = ~err
        mod, row, col = (e.words >> 20) & 0x7FF, (e.words >> 12) & 0xFF, (e.words >> 3) & 0x1FF
        assert np.all(mod[v] < e.n_modules) and np.all(row[v] < 160) and np.all(col[v] < 416)
        assert np.all(np.diff(mod[v].astype(np.int64)) >= 0)                 # module-grouped (A5)
        assert np.all((e.words[v] & 7) == 0) and np.all((e.words[err] & 7) != 0)   # A1
        key = (mod[v].astype(np.int64) << 20) | (row[v] << 10) | col[v]
        assert len(np.unique(key)) == key.shape[0]                           # no duplicate pixels (A6)
        assert e.adc[v].min() >= 10 and e.adc[v].max() <= 255


def test_config3_hot_modules_and_config4_occupancy():
    e = wl.make_event(3, 0)
    v = (e.words >> 31) == 0
    cnt = np.bincount(((e.words >> 20) & 0x7FF)[v], minlength=1856)
    assert 3.3 < cnt[:96].mean() / cnt[96:].mean() < 4.7                    # 4x density (A16)
    e = wl.make_event(4, 0, n_modules=8)
    v = (e.words >> 31) == 0
    cnt = np.bincount(((e.words >> 20) & 0x7FF)[v], minlength=8)
    assert np.all(cnt >= 6656) and np.all(cnt < 6656 + 200)                 # 10 % occupancy


def test_calibration_distributions():
    c = wl.make_calib(1)
    assert c.n_modules == 1856 and c.gain.dtype == np.float32
    assert abs(c.gain.mean() - 80) < 0.5 and abs(c.gain.std() - 5) < 0.4
    assert abs(c.pedestal.mean()) < 15 and abs(c.pedestal.std() - 200) < 12
    assert np.all((c.gain > 0) & (c.gain < 128))
