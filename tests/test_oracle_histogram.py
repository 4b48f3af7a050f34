"""O9 / reading R10: the oracle's histogram rule against numpy on values away from the bin edges, and the edge rules."""
import numpy as np

import oracle


def test_histogram_matches_numpy_and_edge_rules():
    rng = np.random.default_rng(5)
    x = rng.normal(0.9, 0.05, 200_000)
    st = (rng.random(x.size) < 0.1).astype(np.int32)          # 10 % censored (status 1): not counted
    lo, hi, nb = 0.0, 1.05, 1000
    c = oracle.histogram(x, st, lo, hi, nb)
    sel = x[st == 0]
    ref, _ = np.histogram(sel[(sel >= lo) & (sel < hi)], bins=nb, range=(lo, hi))
    assert c[0] == np.sum(sel < lo) and c[-1] == np.sum(sel >= hi)
    assert c.sum() == sel.size
    # numpy computes edges differently (linspace); values within 1e-12 of an edge may differ -- allow only those
    diff = np.abs(c[1:-1].astype(np.int64) - ref)
    assert diff.sum() <= 4
    # edge rules: x == lo -> first bin; x == hi -> "over"; just below hi -> last bin; NaN never counted
    e = oracle.histogram(np.array([lo, hi, np.nextafter(hi, 0), -1e-300, np.nan, 0.5 * (lo + hi)]), None, lo, hi, 10)
    assert e[1] == 1 and e[-1] == 1 and e[10] == 1 and e[0] == 1 and e.sum() == 5 and e[6] == 1
    # accumulation into an existing array
    c2 = oracle.histogram(x, st, lo, hi, nb, counts=c.copy())
    assert np.array_equal(c2, 2 * c)
