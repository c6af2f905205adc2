"""Writes tests/golden/tiny_sequence_scores.txt: the oracle's per-sequence outputs on the `tiny`
config (BASELINE.json configs[0], seed 1001).  Calls only `oracle/` and the input generator.

The paper prints no worked numeric example of c(i), C(tau) or GC, so this
fixture is a regression guard for the oracle + generator pair, not a paper value; the pins that
tie the oracle to the mathematics are in tests/test_oracle_pins.py.

Run from the repo root:  python tests/golden/make_golden.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import sq_oracle as O  # noqa: E402
import workloads  # noqa: E402


def main():
    inp = workloads.make_inputs(workloads.CONFIGS["tiny"])
    out = O.score(inp["H"], inp["W"], inp["targets"], inp["cu_seqlens"], inp["k"], inp["window"])
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_sequence_scores.txt")
    with open(path, "w") as f:
        f.write("# oracle v%d on workloads.CONFIGS['tiny'] (seed 1001, k=5, window=16); Eq. 4 PAPER.md:160\n" % O.ORACLE_VERSION)
        f.write("# seq  length  mean_target_logprob  mean_entropy  mean_conf(C(tau))  min_window_mean_conf\n")
        cu = inp["cu_seqlens"].tolist()
        for b in range(inp["B"]):
            f.write("%d %d %.15e %.15e %.15e %.15e\n" % (
                b, cu[b + 1] - cu[b], out["seq_mean_logprob"][b], out["seq_mean_entropy"][b],
                out["seq_mean_conf"][b], out["seq_min_window_conf"][b]))
    print("wrote", path)


if __name__ == "__main__":
    main()
