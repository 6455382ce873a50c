"""host logic of tests/run_full_parity.py: the broken-set comparator must see a single differing directed bond"""
import importlib.util
import os

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _tool():
    spec = importlib.util.spec_from_file_location("run_full_parity", os.path.join(ROOT, "tests", "run_full_parity.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_broken_keys_match_the_plain_set_and_see_one_differing_bond():
    t = _tool()
    rng = np.random.default_rng(3)
    n = 57
    rows = [np.sort(rng.choice(n, size=rng.integers(0, 9), replace=False)) for _ in range(n)]   # some rows empty
    rowptr = np.concatenate([[0], np.cumsum([len(r) for r in rows])]).astype(np.int64)
    col = np.concatenate(rows).astype(np.int32)
    broken = rng.random(col.size) < 0.3
    keys = t._broken_keys(n, rowptr, col, broken)
    plain = sorted(i * n + int(j) for i in range(n) for p, j in enumerate(rows[i]) if broken[rowptr[i] + p])
    assert keys.dtype == np.int64 and keys.tolist() == plain
    # the same family stored in another order inside the rows (the library's rows are unordered) gives the same keys
    perm = np.concatenate([rowptr[i] + rng.permutation(len(rows[i])) for i in range(n)]).astype(np.int64)
    assert np.array_equal(t._broken_keys(n, rowptr, col[perm], broken[perm]), keys)
    # one flipped bond is one key of difference
    other = broken.copy()
    other[col.size // 2] ^= True
    k2 = t._broken_keys(n, rowptr, col, other)
    assert np.setxor1d(keys, k2, assume_unique=True).size == 1
    # keys do not collide for the largest config (i * n + j < 2^63)
    assert 3144000 * 3144000 < 2 ** 62
