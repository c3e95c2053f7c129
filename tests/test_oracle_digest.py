"""The oracle's arithmetic is frozen by a digest written by tests/golden/make_oracle_digest.py
(a committed script that calls only oracle/)."""
import importlib.util
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_digest_unchanged(oracle_mod):
    spec = importlib.util.spec_from_file_location("make_oracle_digest", os.path.join(HERE, "golden", "make_oracle_digest.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    stored = {}
    with open(os.path.join(HERE, "golden", "oracle_digest.txt")) as f:
        for line in f:
            if not line.startswith("#"):
                name, sha, pairs, coll, rounds = line.split()
                stored[name] = (sha, int(pairs), int(coll), int(rounds))
    for name, mk in mod.CASES.items():
        w, steps = mk()
        assert mod.digest(w, steps) == stored[name], name
