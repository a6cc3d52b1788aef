#!/usr/bin/env python
"""Writes tests/golden/thermalised_<cfg>_seed<s>.txt: the vertex configuration the CPU ORACLE (mode T1)
reaches after `sweeps` sweeps from reset, so that GPU parity tests can start both sides from a
thermalised (well-conditioned) state without minutes of CPU work per test run.

Calls only oracle/ and ctaux_workloads/ (never the CUDA path).  Usage:
    python tests/golden/make_thermalised.py cfg3_4x4_b10 0 40
    python tests/golden/make_thermalised.py cfg4_6x6_b20 0 25
File format: header lines `# key value`, then one line per vertex in list order:
    id site tau(float.hex) spin
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from ctaux_workloads import get_config, table_for  # noqa: E402
from oracle.ctaux_oracle import T1, OracleWalker  # noqa: E402


def main():
    name, seed, sweeps = sys.argv[1], int(sys.argv[2]), int(sys.argv[3])
    cfg = get_config(name)
    o = OracleWalker.from_config(cfg, table_for(cfg), seed, T1)
    o.reset(cfg["init_k"])
    for s in range(sweeps):
        o.sweep(1)
        print(f"sweep {s + 1}/{sweeps}: k = {o.k}", flush=True)
    c = o.config()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"thermalised_{name}_seed{seed}.txt")
    with open(path, "w") as f:
        f.write(f"# config {name}\n# seed {seed}\n# sweeps {sweeps}\n# k {o.k}\n# next_id {o.next_id}\n# p {o.p}\n# sign {o.sign}\n")
        for i in range(o.k):
            f.write(f"{int(c['id'][i])} {int(c['site'][i])} {float(c['tau'][i]).hex()} {int(c['spin'][i])}\n")
    print("wrote", path)


if __name__ == "__main__":
    main()
