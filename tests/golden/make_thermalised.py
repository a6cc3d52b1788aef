#!/usr/bin/env python
"""Writes tests/golden/thermalised_<cfg>_seed<s>.txt: the vertex configuration the CPU ORACLE (mode T1)
reaches after `sweeps` sweeps from reset, so that GPU parity tests can start both sides from a
thermalised (well-conditioned) state without minutes of CPU work per test run.

Calls only oracle/ and ctaux_workloads/ (never the CUDA path).  Usage:
    python tests/golden/make_thermalised.py cfg3_4x4_b10 0 40
    python tests/golden/make_thermalised.py cfg4_6x6_b20 0 25
    python tests/golden/make_thermalised.py cfg5_6x6_b40 1 30      # ~1.5 h of one core
If the file already exists with FEWER sweeps, the chain is continued from it (same seed, same proposal counter:
the oracle's chain does not depend on where it is interrupted -- T1 re-inverts N at every sweep start anyway), so
the result is the configuration after `sweeps` sweeps from reset either way.
File format: header lines `# key value`, then one line per vertex in list order:
    id site tau(float.hex) spin
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

from ctaux_workloads import get_config, table_for  # noqa: E402
from oracle.ctaux_oracle import T1, OracleWalker  # noqa: E402


def write(path, name, seed, sweeps, o):
    c = o.config()
    tmp = path + ".tmp"
    with open(tmp, "w") as f:
        f.write(f"# config {name}\n# seed {seed}\n# sweeps {sweeps}\n# k {o.k}\n# next_id {o.next_id}\n# p {o.p}\n# sign {o.sign}\n")
        for i in range(o.k):
            f.write(f"{int(c['id'][i])} {int(c['site'][i])} {float(c['tau'][i]).hex()} {int(c['spin'][i])}\n")
    os.replace(tmp, path)


def main():
    name, seed, sweeps = sys.argv[1], int(sys.argv[2]), int(sys.argv[3])
    cfg = get_config(name)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"thermalised_{name}_seed{seed}.txt")
    o = OracleWalker.from_config(cfg, table_for(cfg), seed, T1)
    done = 0
    if os.path.exists(path):
        from parity_helpers import load_thermalised
        meta = dict(line.split()[1:3] for line in open(path) if line.startswith("#"))
        if int(meta["sweeps"]) < sweeps:
            c0, next_id, p0 = load_thermalised(name, seed)
            o.set_state(c0["site"], c0["tau"], c0["spin"], c0["id"], next_id, p0)
            done = int(meta["sweeps"])
            print(f"continuing from {path}: {done} sweeps, k = {o.k}", flush=True)
    if done == 0:
        o.reset(cfg["init_k"])
    for s in range(done, sweeps):
        o.sweep(1)
        print(f"sweep {s + 1}/{sweeps}: k = {o.k}", flush=True)
        if (s + 1) % 5 == 0 or s + 1 == sweeps:
            write(path, name, seed, s + 1, o)     # checkpoint: a killed run can be continued
    print("wrote", path)


if __name__ == "__main__":
    main()
