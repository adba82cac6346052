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
