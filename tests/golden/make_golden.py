"""Writes tests/golden/oracle_schedules.txt: digests of the ORACLE's schedules at sizes where re-running
the oracle inside the GPU suite would take minutes to hours (BASELINE.json configs 4 and 5 at full size,
the three relay modes).  Calls only oracle/ and workloads/ -- never the CUDA path.  The GPU parity tests
(tests/test_parity_gpu.py, test_full_size_*_digest) compare the CUDA schedule's digest with these lines.

    python tests/golden/make_golden.py                 # every case below, one after another
    python tests/golden/make_golden.py cfg4:dynamic    # one case (cases may run in parallel processes)

Line format:  case seed transfers time_ps events wants_total sha256(records, canonical order, 32 B each)
Oracle times on this container (one core): cfg4 thin 10 s, bfs 20 s, dynamic 15 min; cfg5 thin 3 min,
bfs ~10 min, dynamic several hours.
"""
import fcntl
import hashlib
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
import workloads as wl  # noqa: E402

OUT = os.path.join(HERE, "oracle_schedules.txt")
RELAYS = {"thin": oracle.RELAY_THIN if hasattr(oracle, "RELAY_THIN") else 0, "dynamic": oracle.RELAY_DYNAMIC,
          "bfs": oracle.RELAY_BFS}
CONFIGS = {"cfg4": wl.config4, "cfg5": wl.config5}
CASES = [f"{c}:{r}" for c in CONFIGS for r in RELAYS]
HEADER = "# written by tests/golden/make_golden.py from oracle/ only; see that file's docstring\n"


def digest(transfers) -> str:
    return hashlib.sha256(transfers.tobytes()).hexdigest()


def run_case(case: str) -> str:
    cfg, relay = case.split(":")
    p = CONFIGS[cfg](0)
    s = oracle.synthesize(*p.args(), relay=RELAYS[relay])
    line = f"{case} {p.seed} {len(s.transfers)} {s.time_ps} {s.events} {s.wants_total} {digest(s.transfers)}\n"
    sys.stdout.write(f"{line.strip()}  ({s.seconds:.1f} s)\n")
    sys.stdout.flush()
    return line


def merge(line: str) -> None:
    """replace or add the line of one case (several processes may finish at once)"""
    with open(OUT, "a+") as f:
        fcntl.flock(f, fcntl.LOCK_EX)
        f.seek(0)
        old = [ln for ln in f.readlines() if not ln.startswith("#")]
        key = line.split()[0]
        keep = [ln for ln in old if ln.split()[0] != key]
        keep.append(line)
        keep.sort(key=lambda ln: CASES.index(ln.split()[0]) if ln.split()[0] in CASES else len(CASES))
        f.seek(0)
        f.truncate()
        f.write(HEADER)
        f.writelines(keep)


def main():
    for case in (sys.argv[1:] or CASES):
        if case not in CASES:
            raise SystemExit(f"unknown case {case}; one of {CASES}")
        merge(run_case(case))


if __name__ == "__main__":
    main()
