"""Test helper: tolerance policy of the GPU-vs-oracle parity tests and the record of what was achieved.

Tolerance:  tol = min(max(nominal, FLOOR_FACTOR * floor), cap)
  nominal  BASELINE.json north_star: log Z relative 1e-10, conditionals absolute 1e-9, log q relative 1e-9
  floor    the ORACLE's own rounding-noise floor for that case (tests/noise_floor.py: one rounding error of
           norm-wise noise per row injected into the oracle's build); a reading, recorded per case
  cap      a hard ceiling: whatever the floor says, nothing passes beyond 100 x nominal
Every comparison goes through `check`, which appends one JSON line (case, quantity, achieved deviation, nominal,
floor, tolerance used and which term was active) to gpurun_out/parity_report.jsonl (or $TNMC_PARITY_REPORT) and
then asserts.  profiles/parity_r2.md is the table made from that file.
"""
import json
import os

FLOOR_FACTOR = 20.0
CAP_FACTOR = 100.0
_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _path():
    p = os.environ.get("TNMC_PARITY_REPORT")
    if p:
        return p
    d = os.path.join(_ROOT, "gpurun_out")
    os.makedirs(d, exist_ok=True)
    return os.path.join(d, "parity_report.jsonl")


def tolerance(nominal, floor):
    """(tol, active term)"""
    wide = FLOOR_FACTOR * float(floor)
    if wide <= nominal:
        return nominal, "nominal"
    cap = CAP_FACTOR * nominal
    return (wide, "floor") if wide <= cap else (cap, "cap")


def record(**kw):
    with open(_path(), "a") as f:
        f.write(json.dumps(kw, default=float) + "\n")


def check(case, quantity, achieved, nominal, floor=0.0, do_assert=True, **extra):
    tol, term = tolerance(nominal, floor)
    ok = bool(achieved <= tol)
    record(case=case, quantity=quantity, achieved=float(achieved), nominal=float(nominal), floor=float(floor),
           tol=float(tol), term=term, ok=ok, **extra)
    if do_assert:
        assert ok, f"{case}: {quantity} deviates by {achieved:.3e} > tol {tol:.3e} ({term}; nominal {nominal:.1e}, floor {floor:.2e})"
    return ok


def table(path=None):
    """markdown summary of a parity_report.jsonl: per (config/beta group, quantity) the worst and median achieved
    deviation, the tolerance terms that were active and the count of failures.
        python tests/parity_report.py [gpurun_out/parity_report.jsonl] > profiles/parity_r2.md"""
    import collections
    import statistics
    rows = [json.loads(ln) for ln in open(path or _path())]
    groups = collections.OrderedDict()
    for r in rows:
        case = r["case"]
        key = (case.split(" d=")[0] + (" " + case.split(" prec=")[1] if " prec=" in case else ""), r["quantity"])
        groups.setdefault(key, []).append(r)
    out = ["| case | quantity | n | worst achieved | median | nominal | tolerance terms used (count) | worst tol | failures |",
           "|---|---|---|---|---|---|---|---|---|"]
    for (case, qty), rs in groups.items():
        if qty == "chains":
            n = sum(r["n"] for r in rs)
            out.append(f"| {case} | chains bit-identical | {n} | {sum(r['identical'] for r in rs)} identical, "
                       f"{sum(r['near_threshold'] for r in rs)} near a threshold | | | | | {sum(1 for r in rs if not r['ok'])} |")
            continue
        ach = [r["achieved"] for r in rs]
        terms = collections.Counter(r["term"] for r in rs)
        out.append(f"| {case} | {qty} | {len(rs)} | {max(ach):.2e} | {statistics.median(ach):.2e} | {rs[0]['nominal']:.0e} | "
                   + ", ".join(f"{k} ({v})" for k, v in sorted(terms.items())) + f" | {max(r['tol'] for r in rs):.2e} | {sum(1 for r in rs if not r['ok'])} |")
    return "\n".join(out)


if __name__ == "__main__":
    import sys
    print(table(sys.argv[1] if len(sys.argv) > 1 else None))
