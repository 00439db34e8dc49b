"""Summarise gpurun_out/parity_report.jsonl (written by `pytest -m gpu`, tests/parity_util.record) as a markdown table:
per test, the worst achieved error per class of series against its bar, and the worst fp64 floor of the oracle's own
double build on the same inputs.

    python -m pytest tests -m gpu -q && python tests/parity_summary.py > profiles/rNN_parity.md
"""
import collections
import json
import os
import re
import sys

ROOT = os.environ.get("GRAFT_REPO_ROOT", os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def klass(series):
    s = str(series)
    if s in ("A", "E", "T"):
        return s
    if s.startswith("XYZ"):
        return "X,Y,Z"
    if s.startswith("y"):
        return "links"
    return s


def main(path=None):
    path = path or os.path.join(ROOT, "gpurun_out", "parity_report.jsonl")
    rows = [json.loads(l) for l in open(path) if l.strip()]
    by = collections.OrderedDict()
    for r in rows:
        pooled = r.get("window") == "pooled"
        per_window = r.get("window") is not None and not pooled
        label = re.sub(r"/source/\d+", "/per source", "/".join(r.get("label", [])))   # sources of a batch share a row
        key = (r.get("test", "?"), label, "window" if per_window else "case")
        d = by.setdefault(key, {})
        c = klass(r.get("series"))
        e = d.setdefault(c, {"err": 0.0, "floor": 0.0, "bar": r.get("bar"), "n": 0})
        e["err"] = max(e["err"], r.get("err") or 0.0)
        fl = r.get("floor", r.get("floor_own_norm"))
        e["floor"] = max(e["floor"], fl or 0.0)
        e["bar"] = max(e["bar"] or 0.0, r.get("bar") or 0.0)
        e["n"] += 1
    print("# GPU parity against the long-double oracle (relative L2; `case` rows: the north-star metric over the whole")
    print("# valid range or pooled over the sampled windows; `window` rows: single sampled windows against their own norm)")
    print()
    print("records: %d, source: %s" % (len(rows), os.path.relpath(path, ROOT)))
    print()
    print("| test | label | kind | series | cases | worst error | worst fp64 floor of the oracle | bar |")
    print("|---|---|---|---|---|---|---|---|")
    worst = collections.defaultdict(float)
    for (test, label, kind), d in by.items():
        for c, e in d.items():
            print("| %s | %s | %s | %s | %d | %.2e | %s | %.0e |" % (test.replace("tests/", ""), label, kind, c, e["n"], e["err"],
                                                                 ("%.2e" % e["floor"]) if e["floor"] else "-", e["bar"]))
            if kind == "case":
                worst[c] = max(worst[c], e["err"] / e["bar"] if e["bar"] else 0.0)
    print()
    print("worst error / bar over the `case` rows: " + ", ".join("%s %.2f" % (c, v) for c, v in worst.items()))


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else None)
