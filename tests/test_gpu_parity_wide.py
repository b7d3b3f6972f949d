"""GPU parity, second part: stress inputs (clustered vertices, where the connected sum cancels hardest), the
shifted-uniform mode (COS_BUILD_UNIFORM_SHIFT; Eq. 33), and wider samples of the two n = 10 BASELINE
configurations at full size in the launch configuration bench.py times.  Bound everywhere: |GPU - oracle| <= 1e-10 * M."""
import multiprocessing as mp
import os

import numpy as np
import pytest

import oracle
from cos_workloads import draw_clustered_vertices, draw_vertices, get_config, random_matrices
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


def _pool():
    return mp.get_context("fork").Pool(min(16, os.cpu_count() or 1))


def _run(cos, w, v, flags=0, shifts="workload"):
    """tabulate + evaluate workload `w` on vertices `v` -> (G numpy [n_blocks*d*d, B], out numpy [n_out, B])."""
    import torch
    table = table_for(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    sig = w.sigmas if shifts == "workload" else shifts
    h = cos.cos_build_ex(w.n, w.n_flavors, w.lattice, sig, w.n if w.all_subsets else 0, flags)
    try:
        G = torch.empty((table.n_blocks * w.d * w.d, w.batch), dtype=torch.float64, device="cuda")
        cos.cos_tabulate(tab, w.n, torch.from_numpy(v["sites"]).cuda(), torch.from_numpy(v["tau"]).cuda(), w.batch, G)
        out = torch.full((cos.cos_info(h, "n_out"), w.batch), float("nan"), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, G, w.batch, out)
        torch.cuda.synchronize()
        return G.cpu().numpy(), out.cpu().numpy()
    finally:
        cos.cos_free(h)
        cos.cos_tab_free(tab)


# ------------------------------------------------------------------------------------------------ stress inputs
@pytest.mark.parametrize("n", [6, 8])
def test_clustered_vertices_uniform_all_subsets(cos, n, capsys):
    """cfg2-shaped (square, SU(2), all subsets) with every configuration's vertices within +-1 site and beta/50 in time
    (SURVEY 8(d) stress input): against the two-determinant route O2a (binary128) on every subset of every
    configuration.  Reports how hard the sums cancel (min |C| / M)."""
    w = get_config(2).scaled(n=n, batch=48 if n == 8 else 96)
    v = draw_clustered_vertices(w)
    G, got = _run(cos, w, v)
    Gh = G.reshape(n, n, w.batch)
    ratio = []
    for c in range(w.batch):
        A = np.ascontiguousarray(Gh[:, :, c])
        ref = oracle.o2a_twospin(A, A)
        M = oracle.o3_uniform(A, 2, 0.0, True, absolute=True)
        assert np.all(np.isfinite(got[:, c]))
        assert np.all(np.abs(got[:, c] - ref) <= TOL * M), (c, (np.abs(got[:, c] - ref) / M).max())
        ratio.append(np.abs(ref[-1]) / M[-1])
    with capsys.disabled():
        print("\n[stress uniform n=%d] full-order |C|/M: min %.2e median %.2e" % (n, min(ratio), np.median(ratio)))
    # the stress input does cancel harder than uniform draws (|C|/M ~ 0.03-0.7 there)
    assert np.median(ratio) < 0.05


def _o2b_and_scale(task):
    A, sig = task
    return oracle.o2b_polynomial(A, sig), oracle.o3_alg3(A, sig, absolute=True)


@pytest.mark.parametrize("n", [6, 8])
def test_clustered_vertices_three_flavours(cos, n, capsys):
    """cfg4-shaped (square, three flavours, non-uniform shifts, SB-CoS), clustered vertices, all subsets at n = 6 and
    the full-order value at n = 8: against the polynomial route Eq. 34-38 (binary128); M = Algorithm 3 on absolute
    values."""
    w = get_config(4).scaled(n=n, batch=40 if n == 6 else 16, all_subsets=(n == 6))
    v = draw_clustered_vertices(w)
    G, got = _run(cos, w, v)
    Gh = G.reshape(3, n, n, w.batch)
    tasks = [(np.ascontiguousarray(Gh[..., c]), w.sigmas) for c in range(w.batch)]
    with _pool() as pool:
        res = pool.map(_o2b_and_scale, tasks, chunksize=1)
    ratio = []
    for c, (ref, M_full) in enumerate(res):
        if w.all_subsets:
            M = oracle.connected_reference(tasks[c][0], n, 1, 3, w.sigmas, False, True, tier="o3", absolute=True)
            assert np.all(np.abs(got[:, c] - ref) <= TOL * M), (c, (np.abs(got[:, c] - ref) / M).max())
        else:
            assert abs(got[0, c] - ref[-1]) <= TOL * M_full, (c, abs(got[0, c] - ref[-1]) / M_full)
        ratio.append(abs(ref[-1]) / M_full)
    with capsys.disabled():
        print("\n[stress SB n=%d] full-order |C|/M: min %.2e median %.2e" % (n, min(ratio), np.median(ratio)))


# ------------------------------------------------------------------------------------------------ shifted-uniform mode
@pytest.mark.parametrize("n,nf,all_subsets", [(1, 2, True), (2, 3, True), (3, 2, True), (4, 3, False), (5, 2, True)])
def test_uniform_shift_vs_bruteforce(cos, n, nf, all_subsets):
    """Uniform CoS with a counterterm (one block, loop factor N_f, true one-cycle A[v][v] + sigma/N_f; PAPER.md:431,
    reading G12) against the definition O1 and against the printed recurrence O3-uniform(sigma), n = 1 included (the
    shift-shift term of Eq. 83 is absent)."""
    import torch
    B = 35 if n < 5 else 3
    sg = 0.37 if n % 2 else -0.55
    G = random_matrices(4000 + 10 * n + nf, 1, n, B, scale=0.8)
    h = cos.cos_build_ex(n, nf, cos.COS_LATTICE_SQUARE, [sg], n if all_subsets else 0, cos.COS_BUILD_UNIFORM_SHIFT)
    try:
        assert cos.cos_info(h, "n_blocks") == 1
        out = torch.empty((cos.cos_info(h, "n_out"), B), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, torch.from_numpy(G.reshape(-1, B)).cuda(), B, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
    finally:
        cos.cos_free(h)
    for c in range(B):
        A = np.ascontiguousarray(G[..., c])
        if all_subsets:
            ref = oracle.o1_all_subsets(A, nf, [sg], sb=False)
            M = oracle.o1_all_subsets(A, nf, [sg], sb=False, absolute=True)
            rec = oracle.o3_uniform(A[0], nf, sg, True)
        else:
            ref = np.array([oracle.o1_connected(A, nf, [sg], sb=False)])
            M = np.array([oracle.o1_connected(A, nf, [sg], sb=False, absolute=True)])
            rec = oracle.o3_uniform(A[0], nf, sg, False)
        assert np.all(np.abs(got[:, c] - ref) <= TOL * M), (c, got[:, c], ref)
        assert np.all(np.abs(got[:, c] - rec) <= TOL * M), (c, got[:, c], rec)


def test_uniform_shift_reductions_n8(cos):
    """n = 8, all 255 subsets, tabulated propagators: (i) two flavours: uniform CoS with shift sigma = two-determinant
    route with sigma_up = sigma_dn = sigma (Eq. 49-50 / O2a'); (ii) Eq. 33: SB-CoS with equal blocks and equal shifts
    returns the uniform value with the same sigma, three flavours; (iii) sigma = 0 reproduces the unshifted handle
    bit for bit (the counterterm only adds 0.0 to the staged diagonal)."""
    import torch
    w = get_config(2).scaled(batch=70)
    v = draw_vertices(w)
    sg = 0.3
    G, plain = _run(cos, w, v)
    _, shifted = _run(cos, w, v, flags=cos.COS_BUILD_UNIFORM_SHIFT, shifts=[sg])
    _, zero = _run(cos, w, v, flags=cos.COS_BUILD_UNIFORM_SHIFT, shifts=[0.0])
    assert np.array_equal(zero, plain)
    Gh = G.reshape(w.n, w.n, w.batch)
    for c in (0, 31, 32, 69):
        A = np.ascontiguousarray(Gh[:, :, c])
        ref = oracle.o2a_twospin(A, A, sg, sg)
        M = oracle.o3_uniform(A, 2, sg, True, absolute=True)
        assert np.all(np.abs(shifted[:, c] - ref) <= TOL * M), (c, (np.abs(shifted[:, c] - ref) / M).max())
        assert np.all(np.abs(shifted[:, c] - oracle.o3_uniform(A, 2, sg, True)) <= TOL * M)
    # (ii) three flavours: SB with three copies of the block and sigma_lambda = sigma vs the uniform handle
    w3 = w.scaled(n_flavors=3)
    _, uni3 = _run(cos, w3, v, flags=cos.COS_BUILD_UNIFORM_SHIFT, shifts=[sg])
    G3 = np.ascontiguousarray(np.broadcast_to(G.reshape(1, -1, w.batch), (3, w.n * w.n, w.batch))).reshape(-1, w.batch)
    h = cos.cos_build(w.n, 3, cos.COS_LATTICE_SQUARE, [sg, sg, sg], w.n)
    try:
        out = torch.empty((255, w.batch), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, torch.from_numpy(G3).cuda(), w.batch, out)
        torch.cuda.synchronize()
        sb3 = out.cpu().numpy()
    finally:
        cos.cos_free(h)
    for c in (0, 33, 69):
        A = np.ascontiguousarray(Gh[:, :, c])
        M = oracle.o3_uniform(A, 3, sg, True, absolute=True)
        assert np.all(np.abs(sb3[:, c] - uni3[:, c]) <= 2 * TOL * M), (c, (np.abs(sb3[:, c] - uni3[:, c]) / M).max())
        assert np.all(np.abs(uni3[:, c] - oracle.o3_uniform(A, 3, sg, True)) <= TOL * M)


def test_uniform_shift_argument_checks(cos):
    with pytest.raises(cos.CosError) as ei:
        cos.cos_build_ex(4, 2, cos.COS_LATTICE_SQUARE, None, 0, cos.COS_BUILD_UNIFORM_SHIFT)
    assert ei.value.code == cos.COS_EINVAL
    # uniform mode has no colour limit: seven flavours with a shift
    h = cos.cos_build_ex(3, 7, cos.COS_LATTICE_SQUARE, [0.1], 0, cos.COS_BUILD_UNIFORM_SHIFT | cos.COS_BUILD_HOST_ONLY)
    assert cos.cos_info(h, "n_blocks") == 1
    cos.cos_free(h)


# ------------------------------------------------------------------------------------------------ n = 10 at full size
def _o2b_full(task):
    A, sig = task
    return oracle.o2b_polynomial(A, sig)[-1]


def _m_lower_sb(task):
    """Rigorous lower bound of M for an SB configuration (see test_gpu_parity.M_lower_bound): the uniform sum on
    min_lambda |A_lambda| with N_f colours per cycle, shift terms dropped."""
    A, nf = task
    return oracle.o3_uniform(np.abs(A).min(axis=0), nf, 0.0, False, absolute=True)[0]


def test_config4_full_64_configurations(cos):
    """BASELINE config 4 at full size (n = 10, three flavours, B = 8192, the launch configuration bench.py times): 64
    configurations -- one whole batch tile (lanes 4096..4127), the first and the last tile's ends, and a spread -- against
    the polynomial route Eq. 34-38 in binary128 (process pool; ~14 s per configuration and core)."""
    import torch
    w = get_config(4)
    v = draw_vertices(w)
    G, got = _run(cos, w, v)
    assert np.all(np.isfinite(got))
    cols = sorted(set(range(4096, 4128)) | {0, 1, 31, 32, 8160, 8190, 8191} | set(range(77, 8192, 331)))[:64]
    assert len(cols) == 64
    Gh = G.reshape(3, w.n, w.n, w.batch)
    mats = [np.ascontiguousarray(Gh[..., c]) for c in cols]
    with _pool() as pool:
        refs = pool.map(_o2b_full, [(A, w.sigmas) for A in mats], chunksize=1)
        Ms = pool.map(_m_lower_sb, [(A, 3) for A in mats], chunksize=1)
    for c, ref, M in zip(cols, refs, Ms):
        assert abs(got[0, c] - ref) <= TOL * M, (c, got[0, c], ref, M)


def _uniform3_ref(task):
    A, sg = task
    return oracle.o3_uniform(A, 3, sg, False)[0], oracle.o3_uniform(A, 3, sg, False, absolute=True)[0]


@pytest.mark.parametrize("n", [11, 12])
def test_sb3_square_orders_11_and_12(cos, n, capsys):
    """The top of the order range north_star names ("two and three flavors, orders n = 4-12"): SB-CoS with three
    flavours on the square lattice (Algorithm 3), config-4-shaped tabulated propagators and shifts, at
    n = 11 (6.3 M states) and n = 12 (21.8 M states), 64 configurations = two batch tiles.
      (a) oracle parity, both orders: with the three blocks equal and equal shifts the SB value is the uniform one with
          that shift (Eq. 33) -- the SB program (colours, fan-out, shift closes) against the uniform recurrence O3 of the
          oracle, bound 1e-10 M;
      (b) oracle parity, n = 11, non-uniform blocks and shifts: the polynomial route Eq. 34-38 in binary128 (7^11 terms,
          ~2 core-minutes per configuration) on three configurations, bound 1e-10 M_lower;
      (c) both orders, every configuration: the determinant route on the device in double-double.  That route loses
          log10(R / |C|) of its ~32 digits (include/cos.h), so it is a corroboration, not an oracle; the observed
          agreement (printed) is ~1e-12 relative at n = 11 and ~1e-11 at n = 12 in the median."""
    import torch
    w = get_config(4).scaled(n=n, batch=64, seed=300 + n)
    v = draw_vertices(w)
    G, got = _run(cos, w, v)
    assert got.shape == (1, w.batch) and np.all(np.isfinite(got)) and np.all(got != 0.0)
    Gh = G.reshape(3, n, n, w.batch)
    # (c) device determinant route, double-double
    Gd = torch.from_numpy(G).cuda()
    sub = torch.full(((1 << n) - 1, w.batch), float("nan"), dtype=torch.float64, device="cuda")
    work = torch.empty((cos.cos_det_workspace_bytes(n, 3, cos.COS_DET_DD, w.batch) + 7) // 8, dtype=torch.float64,
                       device="cuda")
    cos.cos_det_eval(n, 3, 3, w.sigmas, cos.COS_DET_DD, Gd, w.batch, sub, work)
    torch.cuda.synchronize()
    det_full = sub[-1].cpu().numpy()
    del sub, work
    rel = np.abs(det_full - got[0]) / np.abs(got[0])
    with capsys.disabled():
        print("\n[sb3 n=%d] DAG vs device det route (dd): median rel %.2e, max rel %.2e" % (n, np.median(rel), rel.max()))
    assert np.all(np.isfinite(det_full))
    # observed on a B200: n = 11 median 5.2e-13, max 1.4e-10; n = 12 median 9.3e-12, max 2.1e-8
    assert np.median(rel) <= (1e-10 if n == 11 else 1e-9) and rel.max() <= (1e-7 if n == 11 else 1e-5), \
        (np.median(rel), rel.max())
    # (a) Eq. 33 reduction against the uniform oracle
    sg = 0.3
    G1 = np.ascontiguousarray(np.broadcast_to(Gh[:1], Gh.shape)).reshape(-1, w.batch)
    h = cos.cos_build(n, 3, cos.COS_LATTICE_SQUARE, [sg, sg, sg], 0)
    try:
        out = torch.empty((1, w.batch), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, torch.from_numpy(G1).cuda(), w.batch, out)
        torch.cuda.synchronize()
        eq = out.cpu().numpy()[0]
    finally:
        cos.cos_free(h)
    cols = [0, 31, 32, 63]
    with _pool() as pool:
        uni = pool.map(_uniform3_ref, [(np.ascontiguousarray(Gh[0, :, :, c]), sg) for c in cols], chunksize=1)
        if n == 11:
            cols_b = [1, 33, 62]
            mats = [np.ascontiguousarray(Gh[..., c]) for c in cols_b]
            refs = pool.map(_o2b_full, [(A, w.sigmas) for A in mats], chunksize=1)
            Ms = pool.map(_m_lower_sb, [(A, 3) for A in mats], chunksize=1)
    for c, (ref, M) in zip(cols, uni):
        assert abs(eq[c] - ref) <= TOL * M, ("Eq. 33 reduction", n, c, eq[c], ref, M)
    if n == 11:
        for c, ref, M in zip(cols_b, refs, Ms):
            assert abs(got[0, c] - ref) <= TOL * M, ("o2b", c, got[0, c], ref, M)


def _honeycomb_uniform_ref(task):
    Gc, n = task
    return oracle.connected_reference(Gc, n, 2, 2, None, True, False, tier="o2a")[0]


def test_honeycomb_uniform_order_11(cos):
    """The largest honeycomb DAG the layer program can address (include/cos.h: 92 M states, largest layer 15,990,424 of
    the 2^24 - 1 a 24-bit destination index allows): uniform CoS with the sublattice sum (Algorithm 2, PAPER.md:517-544;
    mask refinement PAPER.md:77-84, Eq. 4; sum Eq. 54-55) at n = 11, d = 22 endpoints, config-3-shaped tabulated
    propagators without shifts, one batch tile.  Three configurations against the sum over the 2^11 sublattice assignments
    of the two-determinant route O2a (binary128), bound 1e-10 M_lower."""
    from test_gpu_parity import M_lower_bound
    n = 11
    w = get_config(3).scaled(n=n, alphas=None, batch=32, seed=311)
    v = draw_vertices(w)
    G, got = _run(cos, w, v)
    assert got.shape == (1, w.batch) and np.all(np.isfinite(got)) and np.all(got != 0.0)
    Gh = G.reshape(1, w.d, w.d, w.batch)
    cols = [0, 17, 31]
    mats = [np.ascontiguousarray(Gh[..., c]) for c in cols]
    with _pool() as pool:
        refs = pool.map(_honeycomb_uniform_ref, [(A, n) for A in mats], chunksize=1)
    for c, A, ref in zip(cols, mats, refs):
        M = M_lower_bound(A, n, 2, 2, True, n_assign=8, seed=c)
        assert abs(got[0, c] - ref) <= TOL * M, (c, got[0, c], ref, M)


def _cfg3_ref(task):
    Gc, n, sig = task
    return oracle.connected_reference(Gc, n, 2, 2, sig, False, False, tier="o2a")[0]


def test_config3_full_across_workspace_chunks(cos):
    """BASELINE config 3 at full size (honeycomb, n = 10, B = 16384; the default 64 GiB workspace makes cos_eval walk
    the batch in chunks of 18 tiles = 576 configurations; 17 tiles = 544 with the 64 GB of a smaller budget): 12
    configurations in 7 different chunks, both sides of the first chunk boundary (575 / 576, and 543 / 544) and of a later
    one included, against the sum over the 2^10 sublattice assignments of the two-determinant route O2a' (binary128)."""
    w = get_config(3)
    v = draw_vertices(w)
    G, got = _run(cos, w, v)
    assert np.all(np.isfinite(got))
    cols = [0, 543, 544, 575, 576, 5183, 5184, 9000, 12345, 16127, 16128, 16383]
    Gh = G.reshape(2, w.d, w.d, w.batch)
    mats = [np.ascontiguousarray(Gh[..., c]) for c in cols]
    with _pool() as pool:
        refs = pool.map(_cfg3_ref, [(A, w.n, w.sigmas) for A in mats], chunksize=1)
    from test_gpu_parity import M_lower_bound
    for c, A, ref in zip(cols, mats, refs):
        M = M_lower_bound(A, w.n, 2, 2, False, n_assign=4, seed=c)
        assert abs(got[0, c] - ref) <= TOL * M, (c, got[0, c], ref, M)
