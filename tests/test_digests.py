"""tests/golden/digests.json is what tests/golden/make_digests.py writes from the oracle at HEAD: the two small stored cases
are recomputed here (the large ones come from the same script and take the oracle tens of minutes), and the dense -> CSR
conversion behind the hash is checked against a row-by-row loop."""
import importlib.util
import json
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def _md():
    spec = importlib.util.spec_from_file_location("make_digests", os.path.join(HERE, "golden", "make_digests.py"))
    md = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(md)
    return md


def test_dense_to_csr_row_by_row():
    md = _md()
    rng = np.random.default_rng(3)
    flux = rng.integers(-3, 4, size=(1000, 37)).astype(np.int64) * (rng.random((1000, 37)) < 0.2)
    flux[17] = 0
    row_ptr, rxn, val = md.dense_to_csr(flux, chunk=64)
    assert row_ptr[0] == 0 and row_ptr[-1] == len(rxn) == len(val) == np.count_nonzero(flux)
    for r in range(flux.shape[0]):
        cols = [j for j in range(flux.shape[1]) if flux[r, j] != 0]
        assert rxn[row_ptr[r]:row_ptr[r + 1]].tolist() == cols
        assert val[row_ptr[r]:row_ptr[r + 1]].tolist() == [int(flux[r, j]) for j in cols]
    a = md.digest_csr(row_ptr, rxn, val, np.arange(1000, dtype=np.int32))
    val2 = val.copy(); val2[-1] += 1
    assert md.digest_csr(row_ptr, rxn, val2, np.arange(1000, dtype=np.int32))["rows_sha256"] != a["rows_sha256"]
    assert md.digest_csr(row_ptr, rxn, val, np.arange(1000, dtype=np.int32)[::-1])["steps_sha256"] != a["steps_sha256"]


def test_stored_digests_are_the_oracle_at_head(oracle_mod):
    md = _md()
    with open(os.path.join(HERE, "golden", "digests.json")) as fh:
        cases = json.load(fh)["cases"]
    small = [c for c in cases if c["oracle_seconds"] < 30]
    assert len(small) >= 2 and len(cases) > len(small) - 1
    for c in small:
        d = md.oracle_digest(c["workload"], c["frontier_cap"], 4)
        for k in ("rows", "nnz", "rows_sha256", "steps_sha256", "counters", "levels", "n_roots", "params"):
            assert d[k] == c[k], (c["workload"], k)
