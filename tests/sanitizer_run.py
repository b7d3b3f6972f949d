"""Small end-to-end cases for compute-sanitizer (memcheck / racecheck / initcheck / synccheck), one tool per run:

    compute-sanitizer --tool memcheck python tests/sanitizer_run.py

Covers every kernel of libcos_b200.so on inputs small enough for the sanitizer's slowdown: tabulation, the fused small-DAG
kernel (n = 4 uniform, n = 6 three flavours with shifts), the per-layer kernel with and without programmatic dependent
launch (n = 8, all 255 subsets, ragged batch, two workspace chunks), the honeycomb instantiation, the flux weights, the
determinant route in both precisions and the host-buffer pipeline.  Outputs are only checked for finiteness and for
agreement between the paths (parity against the oracle is tests/test_gpu_*.py); the sanitizer's report is the result.
compute-sanitizer is closed on the pool this was developed on (profiles/r02_sanitizers.md), so the same cases also run
against the self-check build of the library (-DCOS_CHECK_BOUNDS, include/cos.h cos_debug_check_failures; NaN-poisoned
workspace): tests/test_gpu_selfcheck.py."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import paper_2507_12349_b200 as cos  # noqa: E402
from cos_workloads import draw_vertices, get_config, random_matrices  # noqa: E402
from cos_workloads.tables import table_for  # noqa: E402


def evaluate(n, nf, lattice, sig, all_subsets, G, flags=0, tune=None, ws_limit=None):
    B = G.shape[-1]
    h = cos.cos_build_ex(n, nf, lattice, sig, n if all_subsets else 0, flags)
    try:
        for k, v in (tune or {}).items():
            cos.cos_set_tuning(h, k, v)
        if ws_limit:
            cos.cos_set_workspace_limit(h, ws_limit)
        out = torch.zeros((cos.cos_info(h, "n_out"), B), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, torch.from_numpy(np.ascontiguousarray(G.reshape(-1, B))).cuda(), B, out)
        torch.cuda.synchronize()
        return out.cpu().numpy()
    finally:
        cos.cos_free(h)


def main():
    torch.cuda.set_device(0)
    # 1. tabulation + fused kernel + host pipeline (cfg1-shaped, ragged batch)
    w = get_config(1).scaled(batch=45)
    table = table_for(w)
    v = draw_vertices(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    G = torch.zeros((w.n * w.n, w.batch), dtype=torch.float64, device="cuda")
    cos.cos_tabulate(tab, w.n, torch.from_numpy(v["sites"]).cuda(), torch.from_numpy(v["tau"]).cuda(), w.batch, G)
    h = cos.cos_build(w.n, 2, w.lattice, None, 0)
    out = torch.zeros((1, w.batch), dtype=torch.float64, device="cuda")
    cos.cos_eval(h, G, w.batch, out)
    out_h = torch.zeros((1, w.batch), dtype=torch.float64)
    cos.cos_eval_host(h, tab, torch.from_numpy(v["sites"]), torch.from_numpy(v["tau"]), w.batch, out_h)
    torch.cuda.synchronize()
    assert torch.equal(out.cpu(), out_h) and bool(torch.isfinite(out_h).all())
    cos.cos_free(h)
    cos.cos_tab_free(tab)
    # 2. fused kernel, three flavours with shifts, all subsets (n = 6) against the per-layer kernels
    sig = [0.2, 0.0, -0.2]
    G6 = random_matrices(11, 3, 6, 37, scale=0.5, diag=-0.4)
    a = evaluate(6, 3, 0, sig, True, G6)
    b = evaluate(6, 3, 0, sig, True, G6, flags=cos.COS_BUILD_NO_FUSED)
    assert np.array_equal(a, b) and np.all(np.isfinite(a))
    # 3. per-layer kernel, n = 8, all subsets, PDL on / off, two chunks
    G8 = random_matrices(12, 1, 8, 70, scale=0.4, diag=-0.45)
    a = evaluate(8, 2, 0, None, True, G8)
    b = evaluate(8, 2, 0, None, True, G8, tune={"pdl": 0, "tiles_per_chunk": 2, "prefetch": 0})
    c = evaluate(8, 2, 0, [0.3], True, G8, flags=cos.COS_BUILD_UNIFORM_SHIFT, tune={"warps_per_cta": 8})
    assert np.array_equal(a, b) and np.all(np.isfinite(c))
    # 4. honeycomb (d = 2n, long rows), SB two flavours, n = 5 per-layer
    G5 = random_matrices(13, 2, 10, 33, scale=0.4, diag=-0.4)
    a = evaluate(5, 2, 1, [0.3, -0.3], False, G5, flags=cos.COS_BUILD_NO_FUSED)
    assert np.all(np.isfinite(a))
    # 5. partial readout set + flux weights
    h = cos.cos_build_orders(6, 2, 0, None, 0b1010100)
    out = torch.zeros((63, 40), dtype=torch.float64, device="cuda")
    G6u = random_matrices(14, 1, 6, 40, scale=0.5)
    cos.cos_eval(h, torch.from_numpy(G6u.reshape(-1, 40)).cuda(), 40, out)
    W = torch.zeros(40, dtype=torch.float64, device="cuda")
    Phi = torch.zeros((63, 40), dtype=torch.float64, device="cuda")
    cos.cos_flux_weights(6, 0b1010100, [0.0] + [1.0] * 6, out, None, 40, W, Phi)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(W).all())
    cos.cos_free(h)
    # 6. determinant route, both precisions, square and honeycomb
    for prec in (cos.COS_DET_FP64, cos.COS_DET_DD):
        Gd = torch.from_numpy(G6.reshape(-1, 37)).cuda()
        work = torch.zeros((cos.cos_det_workspace_bytes(6, 3, prec, 37) + 7) // 8, dtype=torch.float64, device="cuda")
        o = torch.zeros((63, 37), dtype=torch.float64, device="cuda")
        cos.cos_det_eval(6, 3, 3, sig, prec, Gd, 37, o, work)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(o).all())
    Gh = torch.from_numpy(random_matrices(15, 2, 8, 9, scale=0.4).reshape(-1, 9)).cuda()
    work = torch.zeros((cos.cos_det_workspace_bytes(4, 2, cos.COS_DET_DD, 9) + 7) // 8, dtype=torch.float64, device="cuda")
    o = torch.zeros((15, 9), dtype=torch.float64, device="cuda")
    cos.cos_det_eval(4, 2, 2, [0.3, -0.3], cos.COS_DET_DD, Gh, 9, o, work, lattice=cos.COS_LATTICE_HONEYCOMB)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(o).all())
    total, kinds = cos.cos_debug_check_failures()
    print("self-check failures: %d by kind %s (-1 = library built without COS_CHECK_BOUNDS)" % (total, kinds))
    if os.environ.get("COS_EXPECT_SELFCHECK"):
        assert total == 0, (total, kinds)
    print("sanitizer_run: all cases done")


if __name__ == "__main__":
    main()
