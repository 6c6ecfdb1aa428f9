"""Writes tests/golden/covered_pairs.txt: the number of (particle, pixel) pairs with positive thickness in each of the
five BASELINE.json workloads, counted by the oracle alone (oracle.count_covered, bcircle mode).

    python tests/golden/make_covered_pairs.py

These are the units of SURVEY.md section 8(d)'s "algorithmic flops" (one thickness test per true covered pair);
bench.py reads the file for its ALU roofline.  Nothing here calls the CUDA path.
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import oracle as o            # noqa: E402
from workloads import make_config, CONFIG_NAMES   # noqa: E402


def main():
    lines = ["# workload ellipsoid_pairs prism_pairs   (oracle.count_covered, bcircle mode; written by make_covered_pairs.py)"]
    for cfg in sorted(CONFIG_NAMES):
        ne, np_ = o.count_covered(make_config(cfg))
        lines.append(f"{CONFIG_NAMES[cfg]} {ne} {np_}")
        print(lines[-1], flush=True)
    with open(os.path.join(HERE, "covered_pairs.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
