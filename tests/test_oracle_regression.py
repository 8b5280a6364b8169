"""Regression guard of the oracle (NOT a pin: it compares the oracle with stored results of the oracle).  The pins that
fix what the oracle must compute are in tests/test_oracle_{steps,fit,perigee,precision,surfaces}.py; this file only
notices when a change of oracle/ that was meant to leave a code path alone did not.  CPU only."""
import os

import numpy as np


def test_oracle_regression_digests():
    """The oracle's own results on small seeded workloads against the digests a committed, oracle-only script stored
    (tests/golden/make_oracle_regression.py): a refactoring of the oracle that was meant to leave a code path alone must
    leave these sums alone (1e-11: round-off of a re-association, not of a changed formula)."""
    import importlib.util
    here = os.path.dirname(os.path.abspath(__file__))
    spec = importlib.util.spec_from_file_location("make_oracle_regression", os.path.join(here, "golden", "make_oracle_regression.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    stored = {}
    for line in open(os.path.join(here, "golden", "oracle_regression.txt")):
        if line.startswith("#"):
            continue
        t = line.split()
        stored[t[0]] = np.array([float(v) for v in t[1:]])
    assert set(stored) == {c[0] for c in mod.CASES}
    for c in mod.CASES:
        name, vals = mod.digest(*c)
        np.testing.assert_allclose(np.array(vals), stored[name], rtol=1e-11, atol=0, err_msg=name)
