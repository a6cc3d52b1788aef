"""C-ABI boundary on a machine WITHOUT a GPU: the library builds, loads and exports every entry point
include/ctaux.h declares; the ctypes structures match the header byte for byte; host-only calls behave;
compute calls fail loudly (no CPU fallback); the product package never touches the oracle."""
import ctypes as C
import os
import re
import subprocess
import sys
import tempfile

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ctaux.h")
TEST_HEADER = os.path.join(ROOT, "include", "ctaux_testing.h")


def _declared(header=HEADER):
    src = open(header).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ctaux_[a-z_A-Z0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_1901_01047_b200 import binding
    L = binding.load_library()
    names = _declared()
    assert len(names) >= 19
    helpers = _declared(TEST_HEADER)
    missing = [n for n in names + helpers if not hasattr(L, n)]
    assert not missing, missing
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS and include/ctaux.h disagree"
    assert sorted(binding.TEST_EXPORTS) == helpers, "binding.TEST_EXPORTS and include/ctaux_testing.h disagree"
    # every header under include/ is covered
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["ctaux.h", "ctaux_testing.h"]


def test_ctypes_structs_match_the_header():
    from paper_1901_01047_b200 import binding
    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "ctaux.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu\n", sizeof(ctaux_params), sizeof(ctaux_stats), sizeof(ctaux_log_entry),
         offsetof(ctaux_params, workspace), offsetof(ctaux_params, graph_mode), offsetof(ctaux_stats, flops_cand_alg));
  return 0;
}'''
    with tempfile.TemporaryDirectory() as td:
        src = os.path.join(td, "s.c")
        open(src, "w").write(prog)
        exe = os.path.join(td, "s")
        subprocess.check_call(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), src, "-o", exe])
        out = subprocess.check_output([exe]).split()
    sp, ss, sl, ow, of, og = (int(x) for x in out)
    assert C.sizeof(binding._Params) == sp
    assert C.sizeof(binding._Stats) == ss
    assert binding.LOG_DTYPE.itemsize == sl == 48
    assert binding._Params.workspace.offset == ow
    assert binding._Params.graph_mode.offset == of
    assert binding._Stats.flops_cand_alg.offset == og


def _params(**kw):
    from paper_1901_01047_b200 import binding
    p = binding._Params()
    p.Lx, p.Ly, p.beta, p.U, p.K = 2, 2, 10.0, 4.0, 1.0
    p.n_tau, p.delay, p.n_walkers, p.init_k, p.max_k = 512, 16, 4, 41, 128
    p.rebuild_every, p.log_capacity, p.cand_window = 10, 0, 0
    for k, v in kw.items():
        setattr(p, k, v)
    return p


def test_workspace_bytes_is_host_only_and_validates():
    from paper_1901_01047_b200 import binding
    L = binding.load_library()
    n = L.ctaux_workspace_bytes(C.byref(_params()))
    assert n > 4 * 4 * 128 * 128 * 8           # at least the four N buffers of four walkers
    assert L.ctaux_workspace_bytes(C.byref(_params(n_walkers=8))) > n
    for bad in (dict(delay=0), dict(delay=257), dict(n_walkers=0), dict(init_k=200), dict(beta=0.0), dict(K=-1.0),
                dict(Lx=0), dict(max_k=0), dict(n_tau=0), dict(max_k=9000)):
        assert L.ctaux_workspace_bytes(C.byref(_params(**bad))) == 0, bad
    assert L.ctaux_workspace_bytes(None) == 0


def test_error_strings():
    from paper_1901_01047_b200 import binding
    L = binding.load_library()
    seen = {L.ctaux_strerror(c).decode() for c in (0, -1, -2, -3, -4, -5)}
    assert len(seen) == 6 and "ok" in seen
    assert L.ctaux_strerror(-99).decode() == "unknown error"


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_1901_01047_b200 as pkg
    from ctaux_workloads import get_config, table_for
    cfg = get_config(0)
    with pytest.raises(pkg.CtauxError) as ei:
        pkg.Walkers.from_config(cfg, table_for(cfg))
    assert ei.value.code == -3
    # straight through the C ABI as well: a context cannot be created without a device
    L = pkg.load_library()
    t = np.ascontiguousarray(table_for(cfg))
    p = _params(g0_table=t.ctypes.data, workspace=0x1000, workspace_bytes=1 << 40, max_k=64, init_k=9, delay=8, beta=2.0)
    h = C.c_void_p()
    rc = L.ctaux_create(C.byref(p), C.byref(h))
    assert rc == -3 and not h.value
    assert L.ctaux_sweep(None, 1) == -1 and L.ctaux_reset(None, None) == -1


def test_product_package_does_not_import_the_oracle():
    code = ("import sys; import paper_1901_01047_b200, paper_1901_01047_b200.replicas; "
            "bad=[m for m in sys.modules if m == 'oracle' or m.startswith('oracle.')]; print(bad); sys.exit(1 if bad else 0)")
    subprocess.check_call([sys.executable, "-c", code], cwd=ROOT)
    for fn in os.listdir(os.path.join(ROOT, "paper_1901_01047_b200")):
        if fn.endswith(".py"):
            assert "oracle" not in open(os.path.join(ROOT, "paper_1901_01047_b200", fn)).read().replace("no oracle", "")
