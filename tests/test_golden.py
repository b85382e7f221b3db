"""tests/golden/cfg1_oracle_lines.txt (written by tests/golden/make_golden.py from oracle/ only):
the oracle and the generators still reproduce the stored lines."""
import os

import numpy as np

import oracle
import tdma_inputs

HERE = os.path.dirname(os.path.abspath(__file__))


def load_cfg1_golden():
    out = []
    for ln in open(os.path.join(HERE, "golden", "cfg1_oracle_lines.txt")):
        if ln.startswith("#") or not ln.strip():
            continue
        tok = ln.split()
        out.append((int(tok[0]), int(tok[1]), np.array([float.fromhex(t) for t in tok[2:]])))
    return out


def test_oracle_reproduces_cfg1_golden():
    w = tdma_inputs.make_workload("cfg1_tiny")
    x = oracle.solve_y(w.a.numpy(), w.b.numpy(), w.c.numpy(), w.d.numpy())
    gold = load_cfg1_golden()
    assert len(gold) == 4
    for i, k, ref in gold:
        assert ref.shape == (64,)
        assert np.max(np.abs(x[k, :, i] - ref)) <= 1e-15 * np.max(np.abs(ref))
