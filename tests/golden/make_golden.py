"""Writes tests/golden/oracle_schedules.txt: digests of the ORACLE's schedules on the five
BASELINE.json configs (seed 0) and the reduced variants.  Calls only oracle/ and workloads/
(never the CUDA path).  Used by the GPU parity tests where re-running the oracle at full size
would take minutes (config 5: ~4 min single-threaded).

    python tests/golden/make_golden.py [--skip-config5]

Line format:  name seed transfers time_ps events sha256(transfers bytes, canonical order)
"""
import hashlib
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
import workloads as wl  # noqa: E402


def main():
    makers = [wl.config1, wl.config2, wl.config3, wl.config4_small, wl.config5_small, wl.config4]
    if "--skip-config5" not in sys.argv:
        makers.append(wl.config5)
    lines = ["# written by tests/golden/make_golden.py from oracle/ only; see that file's docstring\n"]
    for mk in makers:
        p = mk(0)
        s = oracle.synthesize(*p.args())
        dig = hashlib.sha256(s.transfers.tobytes()).hexdigest()
        line = f"{p.name} {p.seed} {len(s.transfers)} {s.time_ps} {s.events} {dig}\n"
        sys.stdout.write(f"{line.strip()}  ({s.seconds:.1f} s)\n")
        sys.stdout.flush()
        lines.append(line)
    out = os.path.join(HERE, "oracle_schedules.txt")
    if "--skip-config5" in sys.argv and os.path.exists(out):
        # keep an existing config-5 line
        for old in open(out):
            if old.startswith("cfg5_torus32x32"):
                lines.append(old)
    with open(out, "w") as f:
        f.writelines(lines)


if __name__ == "__main__":
    main()
