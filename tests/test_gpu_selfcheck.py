"""Self-check build of the library: libcos_b200.so compiled with -DCOS_CHECK_BOUNDS tests every index the layer kernels
derive from the compiled program against the extent of the array it addresses and poisons the workspace with NaN
(include/cos.h, cos_debug_check_failures).  compute-sanitizer is closed on the pool this was developed on, so this is the
memcheck / initcheck stand-in: tests/sanitizer_run.py (every kernel, fused and per-layer, PDL on and off, chunked
workspace, honeycomb, partial readouts, determinant route, host pipeline) and two BASELINE-shaped workloads must finish
with zero violations and finite outputs."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKLOADS = r"""
import sys, torch
sys.path.insert(0, %r)
import paper_2507_12349_b200 as cos
from cos_workloads import draw_vertices, get_config
from cos_workloads.tables import table_for
assert cos.cos_debug_check_failures()[0] == 0
for cfg, batch in ((4, 96), (2, 200), (5, 40)):
    w = get_config(cfg).scaled(batch=batch)
    table = table_for(w); v = draw_vertices(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    h = cos.cos_build(w.n, w.n_flavors, w.lattice, w.sigmas, w.n if w.all_subsets else 0)
    G = torch.empty((w.n_blocks * w.d * w.d, batch), dtype=torch.float64, device="cuda")
    cos.cos_tabulate(tab, w.n, torch.from_numpy(v["sites"]).cuda(), torch.from_numpy(v["tau"]).cuda(), batch, G)
    out = torch.full((w.n_out, batch), float("nan"), dtype=torch.float64, device="cuda")
    cos.cos_eval(h, G, batch, out)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all()), cfg
    cos.cos_free(h); cos.cos_tab_free(tab)
total, kinds = cos.cos_debug_check_failures()
print("self-check failures after cfg4 / cfg2 / cfg5 shaped runs:", total, kinds)
assert total == 0
"""


def test_selfcheck_build_reports_no_violation(tmp_path):
    import torch
    assert torch.cuda.is_available()
    sys.path.insert(0, ROOT)
    from paper_2507_12349_b200 import build
    import paper_2507_12349_b200 as cos
    assert cos.cos_debug_check_failures()[0] == -1          # the shipped build has the checks compiled out
    lib = build.build(out=str(tmp_path / "libcos_b200_selfcheck.so"), extra=["-DCOS_CHECK_BOUNDS"])
    env = dict(os.environ, COS_B200_LIB=lib, COS_EXPECT_SELFCHECK="1", PYTHONPATH=ROOT)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitizer_run.py")], env=env, capture_output=True,
                       text=True, timeout=1200)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert "self-check failures: 0 " in r.stdout and "all cases done" in r.stdout
    r = subprocess.run([sys.executable, "-c", WORKLOADS % ROOT], env=env, capture_output=True, text=True, timeout=1200)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
