"""Writes tests/golden/oracle_digest.txt: SHA-256 digests of the oracle's state after a few
steps of two small workloads.  Calls only `oracle/` and `workloads/` (never the CUDA path).
The digest guards the oracle's arithmetic against accidental change: any edit that moves a
bit must be justified in its commit message by the PAPER.md passage or DESIGN.md reading.

    python tests/golden/make_oracle_digest.py
"""
import hashlib
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle      # noqa: E402
import workloads   # noqa: E402


def digest(w, steps):
    o = oracle.Oracle.from_workload(w)
    o.step(steps, w.dt, w.sigma)
    h = hashlib.sha256()
    for a in o.particles():
        h.update(a.tobytes())
    c = o.counters()
    return h.hexdigest(), c["pairs"], c["collisions"], c["rounds"]


CASES = {
    "configs0_3steps": lambda: (workloads.make(0), 3),
    "riemann_small_5steps": lambda: (workloads.riemann_small(), 5),
}

if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_digest.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_oracle_digest.py (oracle only): name sha256 pairs collisions rounds\n")
        for name, mk in CASES.items():
            w, steps = mk()
            f.write("%s %s %d %d %d\n" % ((name,) + digest(w, steps)))
    print(open(out).read())
