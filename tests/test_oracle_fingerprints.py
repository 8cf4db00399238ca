"""Tripwire on the oracle's arithmetic (no GPU): tests/golden/oracle_fingerprints.txt was written by
tests/golden/make_oracle_fingerprints.py from oracle/ alone.  A mismatch means the oracle changed; if that is intended,
re-run the script and name the PAPER.md passage / DESIGN.md reading that justifies the change in the commit message."""
import importlib.util
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_output_is_what_it_was():
    spec = importlib.util.spec_from_file_location("make_fp", os.path.join(HERE, "golden", "make_oracle_fingerprints.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    stored = {}
    for line in open(os.path.join(HERE, "golden", "oracle_fingerprints.txt")):
        if line.startswith("#"):
            continue
        name, relax, what, a, b = line.split()
        stored[(name, relax, what)] = (float(a), float(b))
    now = {(n, r, w): (a, b) for n, r, w, a, b in mod.fingerprints()}
    assert set(now) == set(stored)
    for k, (a, b) in now.items():
        sa, sb = stored[k]
        # summation order inside numpy / BLAS may differ between machines: 1e-11 relative on O(1)-weighted sums
        assert abs(a - sa) <= 1e-11 * max(1.0, abs(sa), abs(sb) * 1e3), (k, a, sa)
        assert abs(b - sb) <= 1e-11 * max(abs(sb), 1e-300) + 1e-18, (k, b, sb)
