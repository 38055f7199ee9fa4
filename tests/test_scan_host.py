"""-m "not gpu": the host statistics of the temperature-scan driver (jackknife over blocks)."""
import numpy as np


def test_jackknife_of_a_mean_and_of_a_variance():
    from paper_2301_11735_b200.scan import _jackknife
    rng = np.random.default_rng(7)
    nb = 64
    x = rng.normal(2.0, 0.5, size=(nb, 1000))
    blocks = np.stack([x.mean(axis=1), (x * x).mean(axis=1)], axis=1)          # per-block <x>, <x^2>
    m, em = _jackknife(blocks, lambda v: v[0])
    assert abs(m - x.mean()) < 1e-12
    assert abs(em - blocks[:, 0].std(ddof=1) / np.sqrt(nb)) < 1e-12            # jackknife of a mean = standard error
    var, ev = _jackknife(blocks, lambda v: v[1] - v[0] * v[0])
    assert abs(var - 0.25) < 5 * ev and 0 < ev < 0.01                          # sigma^2 = 0.25 within its error


def test_parse_temperatures():
    from paper_2301_11735_b200.scan import _parse_T
    assert _parse_T("0.1:4.0:41")[0] == 0.1 and len(_parse_T("0.1:4.0:41")) == 41 and abs(_parse_T("0.1:4.0:41")[-1] - 4.0) < 1e-12
    assert _parse_T("0.5,1,2") == [0.5, 1.0, 2.0]
