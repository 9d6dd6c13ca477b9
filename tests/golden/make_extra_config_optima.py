"""Writes tests/golden/extra_config_optima.txt: optimum costs (and a checksum of the optimal strategy) of the three configs
that are not in BASELINE.json, computed by the ORACLE ONLY (oracle/ref.py; nothing under paper_2301_06813_b200/csrc is
loaded).  These are regression values for the oracle -- a change of its arithmetic shows up here and must name the
reading that justifies it -- not values of the paper.  Run from the repo root:

    python tests/golden/make_extra_config_optima.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import ref                                   # noqa: E402
from paper_2301_06813_b200 import configs as cf         # noqa: E402  (seeded input generators only)


def main():
    lines = ["# Written by tests/golden/make_extra_config_optima.py from the oracle alone (DESIGN.md R24-R26).",
             "# configN_dp = optimum cost in ps; configN_strategy_sum = sum over layers of (l + 1) * s_l of the optimal strategy."]
    for k in (6, 7, 8):
        w = cf.CONFIGS[k]()
        T, _, _ = ref.build_tables(w.layers, ref.mesh_of(w), ref.net_of(w))
        dc, ds = ref.chain_dp(T)
        lines.append("config%d_dp = %d" % (k, int(dc[0])))
        lines.append("config%d_strategy_sum = %d" % (k, sum((l + 1) * int(s) for l, s in enumerate(ds[0]))))
    with open(os.path.join(ROOT, "tests", "golden", "extra_config_optima.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
