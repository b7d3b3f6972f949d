"""GPU tests of the host-buffer entry point cos_eval_host (the call bench.py's `e2e` number is measured through), of
the measurement helpers, of cos_reserve / CUDA-graph capture, of the workspace chunking of the per-layer kernels, and of
the argument checks of the binding.  Every comparison against the oracle uses the bound of test_gpu_parity.py:
|GPU - oracle| <= 1e-10 * M (BASELINE.json north_star)."""
import numpy as np
import pytest

import oracle
from cos_workloads import draw_vertices, get_config, random_matrices
from cos_workloads.tables import table_for

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def cos():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    torch.cuda.set_device(0)
    import paper_2507_12349_b200 as cos_mod
    cos_mod.load_library()
    return cos_mod


def _host_inputs(w, pinned):
    import torch
    v = draw_vertices(w)
    sites, tau = torch.from_numpy(v["sites"]), torch.from_numpy(v["tau"])
    out = torch.full((w.n_out, w.batch), float("nan"), dtype=torch.float64)
    if pinned:
        sites, tau, out = sites.pin_memory(), tau.pin_memory(), out.pin_memory()
    return v, sites, tau, out


def _device_reference(cos, w, tab, h, v):
    """tabulate + cos_eval with device-resident inputs: what cos_eval_host must reproduce bit for bit."""
    import torch
    G = torch.empty((w.n_blocks * w.d * w.d, w.batch), dtype=torch.float64, device="cuda")
    cos.cos_tabulate(tab, w.n, torch.from_numpy(v["sites"]).cuda(), torch.from_numpy(v["tau"]).cuda(), w.batch, G)
    out = torch.full((w.n_out, w.batch), float("nan"), dtype=torch.float64, device="cuda")
    cos.cos_eval(h, G, w.batch, out)
    torch.cuda.synchronize()
    return G.cpu().numpy(), out.cpu().numpy()


def test_eval_host_sliced_pipeline_against_oracle(cos):
    """cfg2-shaped (n = 8, all 255 subsets), B = 8237: the output (16.8 MB) is produced in slices whose columns return
    on a second stream while the next slice is evaluated; B is not a multiple of 32 (ragged last tile) nor of the
    slice count.  Every column must equal the device-resident path bit for bit (same kernels, same order), with 1 or
    8 slices, pinned or pageable host buffers; whole slices' worth of sampled columns (both ends of every slice
    boundary) against the two-determinant route O2a on every subset (PAPER.md:491 is the path, Eq. 13-15 the outputs)."""
    w = get_config(2).scaled(batch=8237)
    table = table_for(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    h = cos.cos_build(w.n, w.n_flavors, w.lattice, w.sigmas, w.n)
    try:
        v, sites, tau, out = _host_inputs(w, pinned=True)
        G_ref, dev_out = _device_reference(cos, w, tab, h, v)
        launches0 = cos.cos_info(h, "n_launches")
        cos.cos_eval_host(h, tab, sites, tau, w.batch, out)
        sliced = out.numpy().copy()
        n_launch_sliced = cos.cos_info(h, "n_launches") - launches0
        assert np.array_equal(sliced, dev_out)
        # the call really took the sliced path: one tabulation + n_slices x (fill + 16 layers) launches
        tiles = (w.batch + 31) // 32
        n_slices = min(8, (w.n_out * w.batch * 8) >> 23, tiles)
        assert n_slices > 1 and n_launch_sliced == 1 + n_slices * 17
        # one slice (no second stream), pageable buffers
        cos.cos_set_tuning(h, "host_slices", 1)
        v2, sites_p, tau_p, out_p = _host_inputs(w, pinned=False)
        launches0 = cos.cos_info(h, "n_launches")
        cos.cos_eval_host(h, tab, sites_p, tau_p, w.batch, out_p)
        assert cos.cos_info(h, "n_launches") - launches0 == 1 + 17
        assert np.array_equal(out_p.numpy(), dev_out)
        cos.cos_set_tuning(h, "host_slices", 3)
        out_p.fill_(float("nan"))
        cos.cos_eval_host(h, tab, sites_p, tau_p, w.batch, out_p)
        assert np.array_equal(out_p.numpy(), dev_out)
        # oracle on the columns around every slice boundary and the ragged tail
        cols = {0, 1, 31, 32, w.batch - 1, w.batch - 2, w.batch - 6}
        for i in range(1, n_slices):
            c = (tiles * i // n_slices) * 32
            cols.update({c - 1, c, c + 1})
        Gh = G_ref.reshape(w.n, w.n, w.batch)
        for c in sorted(cols):
            A = np.ascontiguousarray(Gh[:, :, c])
            M = oracle.o3_uniform(A, 2, 0.0, True, absolute=True)
            ref = oracle.o2a_twospin(A, A)
            assert np.all(np.abs(sliced[:, c] - ref) <= TOL * M), (c, np.abs(sliced[:, c] - ref).max())
    finally:
        cos.cos_free(h)
        cos.cos_tab_free(tab)


def test_eval_host_staging_regrowth_and_small_batches(cos):
    """A second call with a larger batch regrows the staging area; batches 1, 31, 33 and 0; SB three flavours n = 5
    against the brute-force definition O1."""
    import torch
    w0 = get_config(4).scaled(n=5, batch=200)
    table = table_for(w0)
    tab = cos.cos_tab_build(w0.lattice, w0.L, table.n_blocks, w0.beta, w0.n_tau, table.data)
    h = cos.cos_build(w0.n, w0.n_flavors, w0.lattice, w0.sigmas, 0)
    try:
        for B in (1, 31, 33, 200, 64):
            w = w0.scaled(batch=B)
            v, sites, tau, out = _host_inputs(w, pinned=(B != 33))
            cos.cos_eval_host(h, tab, sites, tau, B, out)
            G_ref = oracle.tabulate_reference(table, v["sites"], v["tau"])
            got = out.numpy()
            assert np.all(np.isfinite(got))
            for c in sorted({0, B - 1, B // 2}):
                A = np.ascontiguousarray(G_ref[:, :, :, c])
                ref = oracle.o1_connected(A, 3, w.sigmas, sb=True)
                M = oracle.o1_connected(A, 3, w.sigmas, sb=True, absolute=True)
                assert abs(got[0, c] - ref) <= TOL * M, (B, c)
        # batch 0 is a no-op and touches nothing
        out = torch.full((1, 4), 7.0, dtype=torch.float64)
        cos.cos_eval_host(h, tab, torch.zeros((5, 2, 0), dtype=torch.int32), torch.zeros((5, 0), dtype=torch.float64), 0, out)
        assert bool((out == 7.0).all())
        # a table of the wrong shape is refused
        w2 = get_config(1)
        t2 = table_for(w2)
        tab2 = cos.cos_tab_build(w2.lattice, w2.L, t2.n_blocks, w2.beta, w2.n_tau, t2.data)
        v, sites, tau, out = _host_inputs(w0.scaled(batch=8), pinned=False)
        with pytest.raises(cos.CosError) as ei:
            cos.cos_eval_host(h, tab2, sites, tau, 8, out)
        assert ei.value.code == cos.COS_EINVAL
        cos.cos_tab_free(tab2)
    finally:
        cos.cos_free(h)
        cos.cos_tab_free(tab)


def test_profiling_helpers_leave_the_outputs_unchanged(cos):
    """cos_set_profiling / cos_get_layer_times (per-layer CUDA events; they serialise the layers): positive times for
    every launched layer, the evaluation count, cleared records, and bit-identical outputs."""
    import torch
    n, B = 8, 300
    G = random_matrices(91, 1, n, B, scale=0.4, diag=-0.45)
    Gd = torch.from_numpy(G.reshape(-1, B)).cuda()
    h = cos.cos_build(n, 2, cos.COS_LATTICE_SQUARE, None, n)
    try:
        out0 = torch.empty((255, B), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, Gd, B, out0)
        cos.cos_set_profiling(h, True)
        out1 = torch.empty_like(out0)
        for _ in range(3):
            cos.cos_eval(h, Gd, B, out1)
        ms, n_eval = cos.cos_get_layer_times(h)
        assert n_eval == 3 and len(ms) == 2 * n
        assert all(t > 0.0 for t in ms)
        ms2, n2 = cos.cos_get_layer_times(h)                  # cleared by the first call
        assert n2 == 0 and sum(ms2) == 0.0
        cos.cos_set_profiling(h, False)
        out2 = torch.empty_like(out0)
        cos.cos_eval(h, Gd, B, out2)
        torch.cuda.synchronize()
        assert torch.equal(out0, out1) and torch.equal(out0, out2)
    finally:
        cos.cos_free(h)


def test_reserve_makes_eval_capturable_in_a_cuda_graph(cos):
    """After cos_reserve(h, B) a cos_eval with batch <= B only enqueues kernels: the workspace does not change and the
    call can be captured into a CUDA graph and replayed (include/cos.h, cos_eval / cos_reserve)."""
    import torch
    n, nf, B = 7, 3, 257
    sig = [0.2, 0.0, -0.2]
    G = random_matrices(92, nf, n, B, scale=0.5, diag=-0.4)
    Gd = torch.from_numpy(G.reshape(-1, B)).cuda()
    h = cos.cos_build(n, nf, cos.COS_LATTICE_SQUARE, sig, 0)
    try:
        assert cos.cos_info(h, "workspace_bytes") == 0
        assert cos.cos_info(h, "device") == torch.cuda.current_device()
        cos.cos_reserve(h, B)
        ws = cos.cos_info(h, "workspace_bytes")
        tiles = (B + 31) // 32
        assert ws == 2 * cos.cos_info(h, "max_layer_states") * 32 * 8 * tiles
        ref = torch.empty((1, B), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, Gd, B, ref)
        torch.cuda.synchronize()
        assert cos.cos_info(h, "workspace_bytes") == ws
        out = torch.zeros((1, B), dtype=torch.float64, device="cuda")
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            cos.cos_eval(h, Gd, B, out)
        out.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, ref)
        Gd.mul_(0.5)                                          # the graph reads the caller's buffer at replay time
        graph.replay()
        cos.cos_eval(h, Gd, B, ref)
        torch.cuda.synchronize()
        assert torch.equal(out, ref)
        cos.cos_reserve(h, 0)
        with pytest.raises(cos.CosError):
            cos.cos_reserve(h, -1)
    finally:
        cos.cos_free(h)


def test_eval_that_must_grow_the_workspace_fails_cleanly_under_capture(cos):
    """A cos_eval whose batch exceeds what cos_reserve prepared would have to cudaFree + cudaMalloc the workspace; while
    its stream is being captured it must refuse (COS_EINVAL), enqueue nothing and leave the capture usable
    (include/cos.h, cos_eval)."""
    import torch
    n, nf, B, B_big = 7, 2, 64, 256
    G = random_matrices(93, 1, n, B_big, scale=0.5, diag=-0.4)
    Gd = torch.from_numpy(G.reshape(-1, B_big)).cuda()
    Gs = Gd[:, :B].contiguous()
    h = cos.cos_build_ex(n, nf, cos.COS_LATTICE_SQUARE, None, 0, flags=cos.COS_BUILD_NO_FUSED)
    try:
        cos.cos_reserve(h, B)
        assert cos.cos_info(h, "reserved_batch") == B
        ws = cos.cos_info(h, "workspace_bytes")
        ref = torch.empty((1, B), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, Gs, B, ref)
        torch.cuda.synchronize()
        out = torch.zeros((1, B), dtype=torch.float64, device="cuda")
        big = torch.full((1, B_big), float("nan"), dtype=torch.float64, device="cuda")
        launches = cos.cos_info(h, "n_launches")
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            with pytest.raises(cos.CosError) as ei:
                cos.cos_eval(h, Gd, B_big, big)                   # needs 4x the reserved workspace
            assert ei.value.code == cos.COS_EINVAL and "cos_reserve" in str(ei.value)
            assert cos.cos_info(h, "n_launches") == launches      # nothing enqueued
            cos.cos_eval(h, Gs, B, out)                           # the capture goes on
        assert cos.cos_info(h, "workspace_bytes") == ws
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, ref) and bool(torch.isnan(big).all())
        cos.cos_eval(h, Gd, B_big, big)                           # outside a capture the same call grows the workspace
        torch.cuda.synchronize()
        assert cos.cos_info(h, "workspace_bytes") > ws and torch.equal(big[:, :B], ref)
    finally:
        cos.cos_free(h)


@pytest.mark.parametrize("n,nf,sb,all_subsets", [(8, 2, False, True), (7, 3, True, False)])
def test_per_layer_kernels_chunked_workspace(cos, n, nf, sb, all_subsets):
    """Orders above 6 run the per-layer kernels (cos_layer_kernel).  A 1-byte workspace limit makes cos_eval walk the
    batch one 32-configuration tile per chunk, `tiles_per_chunk` two tiles per chunk: same launches per tile, so the
    outputs are bit-identical to the unchunked call; sampled columns against the oracle."""
    import torch
    B = 165                                                    # 6 tiles, ragged
    sig = [0.3, -0.2, 0.1][:nf] if sb else None
    G = random_matrices(93 + n, nf if sb else 1, n, B, scale=0.5, diag=-0.4)
    Gd = torch.from_numpy(G.reshape(-1, B)).cuda()
    outs = []
    for mode in ("plain", "one_tile", "two_tiles"):
        h = cos.cos_build(n, nf, cos.COS_LATTICE_SQUARE, sig, n if all_subsets else 0)
        try:
            assert cos.cos_info(h, "fused") == 0
            if mode == "one_tile":
                cos.cos_set_workspace_limit(h, 1)
            if mode == "two_tiles":
                cos.cos_set_tuning(h, "tiles_per_chunk", 2)
            out = torch.full((cos.cos_info(h, "n_out"), B), float("nan"), dtype=torch.float64, device="cuda")
            l0 = cos.cos_info(h, "n_launches")
            cos.cos_eval(h, Gd, B, out)
            torch.cuda.synchronize()
            chunks = {"plain": 1, "one_tile": 6, "two_tiles": 3}[mode]
            assert cos.cos_info(h, "n_launches") - l0 == chunks * (1 + 2 * n)
            per_tile = 2 * cos.cos_info(h, "max_layer_states") * 32 * 8
            assert cos.cos_info(h, "workspace_bytes") == per_tile * {"plain": 6, "one_tile": 1, "two_tiles": 2}[mode]
            outs.append(out.cpu().numpy())
        finally:
            cos.cos_free(h)
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
    for c in (0, 31, 32, 100, 164):
        A = np.ascontiguousarray(G[..., c])
        if sb:
            ref = oracle.o2b_polynomial(A, sig)[-1:]
            M = np.array([oracle.o3_alg3(np.abs(A), np.abs(sig), absolute=True)])
        else:
            ref = oracle.o2a_twospin(A[0], A[0])
            M = oracle.o3_uniform(A[0], 2, 0.0, True, absolute=True)
        assert np.all(np.abs(outs[0][:, c] - ref) <= TOL * M), (c, np.abs(outs[0][:, c] - ref).max())


def test_binding_rejects_undersized_tensors(cos):
    """The Python binding checks that every tensor holds what the call reads or writes (COS_EINVAL instead of an
    out-of-bounds device access)."""
    import torch
    n, B = 4, 64
    h = cos.cos_build(n, 2, cos.COS_LATTICE_SQUARE, None, n)
    w = get_config(1)
    table = table_for(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    try:
        G = torch.zeros((n * n, B), dtype=torch.float64, device="cuda")
        out = torch.zeros((15, B), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, G, B, out)
        for bad_G, bad_out in ((G[:, : B - 1].contiguous(), out), (G, out[:14].contiguous()),
                               (G.float(), out), (G.cpu(), out)):
            with pytest.raises(cos.CosError) as ei:
                cos.cos_eval(h, bad_G, B, bad_out)
            assert ei.value.code == cos.COS_EINVAL
        sites = torch.zeros((n, 2, B), dtype=torch.int32, device="cuda")
        tau = torch.zeros((n, B), dtype=torch.float64, device="cuda")
        cos.cos_tabulate(tab, n, sites, tau, B, G)
        for args in ((sites[:, :1].contiguous(), tau, G), (sites, tau[: n - 1].contiguous(), G),
                     (sites, tau, G[: n * n - 1].contiguous())):
            with pytest.raises(cos.CosError) as ei:
                cos.cos_tabulate(tab, n, args[0], args[1], B, args[2])
            assert ei.value.code == cos.COS_EINVAL
        with pytest.raises(cos.CosError):
            cos.cos_eval_host(h, tab, sites.cpu(), tau.cpu(), B, torch.zeros((15, B - 1), dtype=torch.float64))
        W = torch.zeros(B, dtype=torch.float64, device="cuda")
        with pytest.raises(cos.CosError):
            cos.cos_flux_weights(n, 0, [0.0] + [1.0] * n, out[:14].contiguous(), None, B, W)
        torch.cuda.synchronize()
    finally:
        cos.cos_free(h)
        cos.cos_tab_free(tab)


def test_tabulate_times_at_and_beyond_the_table_ends(cos):
    """tau = 0 and tau just below beta are bit-exact against the oracle (end nodes of the table, readings G17-G18);
    times outside [0, beta) and non-finite times read no memory outside the table: finite extrapolations / NaN, no fault."""
    import torch
    w = get_config(1).scaled(batch=64)
    table = table_for(w)
    v = draw_vertices(w)
    v["tau"][0, :16] = 0.0
    v["tau"][1, :16] = np.nextafter(w.beta, 0.0)
    v["tau"][2, 16:32] = np.nextafter(w.beta, 0.0)
    v["tau"][3, 16:32] = 0.0
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    try:
        G = torch.empty((w.n * w.n, 64), dtype=torch.float64, device="cuda")
        cos.cos_tabulate(tab, w.n, torch.from_numpy(v["sites"]).cuda(), torch.from_numpy(v["tau"]).cuda(), 64, G)
        torch.cuda.synchronize()
        ref = oracle.tabulate_reference(table, v["sites"], v["tau"])
        assert np.array_equal(G.cpu().numpy(), ref.reshape(-1, 64))
        bad = v["tau"].copy()
        bad[0, 0], bad[1, 1], bad[2, 2], bad[3, 3] = 5.0 * w.beta, -7.0 * w.beta, np.inf, np.nan
        bad[0, 4], bad[1, 4] = 1e300, -1e300
        sites_bad = v["sites"].copy()
        sites_bad[0, 0, 5], sites_bad[1, 1, 5] = 10 ** 6, -(10 ** 6)          # reduced modulo L
        cos.cos_tabulate(tab, w.n, torch.from_numpy(sites_bad).cuda(), torch.from_numpy(bad).cuda(), 64, G)
        torch.cuda.synchronize()
        Gh = G.cpu().numpy()
        assert np.all(np.isfinite(Gh[:, 6:]))
        assert np.array_equal(Gh[:, 6:], ref.reshape(-1, 64)[:, 6:])
        assert np.all(np.isfinite(Gh[:, 5]))
    finally:
        cos.cos_tab_free(tab)
