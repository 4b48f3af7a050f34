"""Pin P1: the oracle's Philox4x32-10 against published known answers and a from-definition
pure-Python implementation (tests/ref_mp.py)."""
import numpy as np

import oracle
from ref_mp import philox4x32_10 as py_philox, philox_block as py_block, read_golden


def test_known_answers_raw():
    rows = [r for r in read_golden("philox_kat.txt") if r[0] == "raw"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r[1:]]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])
        assert py_philox(tuple(v[0:4]), tuple(v[4:6])) == tuple(v[6:10])


def test_known_answers_keyed():
    rows = [r for r in read_golden("philox_kat.txt") if r[0] == "keyed"]
    assert len(rows) == 4
    for r in rows:
        seed, tid, block = int(r[1]), int(r[2]), int(r[3])
        want = tuple(int(x, 16) for x in r[4:8])
        assert oracle.philox_block(seed, tid, block) == want
        assert py_block(seed, tid, block) == want


def test_against_python_random_inputs():
    rng = np.random.default_rng(11)
    for _ in range(300):
        ctr = [int(x) for x in rng.integers(0, 2**32, 4)]
        key = [int(x) for x in rng.integers(0, 2**32, 2)]
        assert oracle.philox4x32_10(ctr, key) == py_philox(tuple(ctr), tuple(key))


def test_keying_uses_all_64_bits():
    # seed hi word, id hi word and block hi word each change the output (reading R1)
    base = oracle.philox_block(7, 9, 3)
    assert oracle.philox_block(7 + 2**32, 9, 3) != base
    assert oracle.philox_block(7, 9 + 2**32, 3) != base
    assert oracle.philox_block(7, 9, 3 + 2**32) != base
    assert oracle.philox_block(7 + 2**32, 9, 3) == py_block(7 + 2**32, 9, 3)
    assert oracle.philox_block(7, 9 + 2**40, 3 + 2**33) == py_block(7, 9 + 2**40, 3 + 2**33)
