"""The oracle against its stored anchors (tests/golden/oracle_anchors.txt, written by tests/golden/make_golden.py from
oracle/ alone): bit for bit.  A failure here means the oracle's arithmetic changed; see tests/golden/README.md."""
import importlib.util
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def load_generator():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_oracle_matches_its_anchors_bit_for_bit():
    stored = {}
    for line in open(os.path.join(HERE, "golden", "oracle_anchors.txt")):
        if line.startswith("#") or not line.strip():
            continue
        key, vals, cite = (p.strip() for p in line.split("|"))
        assert cite, key                                           # every anchor names the passage that defines it
        stored[key] = vals.split()
    now = {key: vals for key, vals, _ in load_generator().anchors()}
    assert sorted(now) == sorted(stored)
    for key in stored:
        assert now[key] == stored[key], key
    assert sum(len(v) for v in stored.values()) == 100              # the fixture as generated: 21 anchors, 100 values
