"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Every test here needs a B200 (`-m gpu`).

Acceptance bound (BASELINE.json north_star): |GPU - oracle| <= 1e-10 * M, M = the same sum evaluated
on |G|, |sigma| with every sign dropped (oracle `absolute=True`).  Where M is too slow to compute
(n >= 10, SB) the test uses the STRICTER bound 1e-10 * M_lower_bound(...) <= 1e-10 * M.
The tabulation step is compared bit for bit (both sides fix the rounding order).
"""
import json
import os

import numpy as np
import pytest

import oracle
from cos_workloads import draw_vertices, get_config, random_matrices
from cos_workloads.tables import table_for

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))
TOL = 1e-10


@pytest.fixture(scope="module")
def cos():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    torch.cuda.set_device(0)
    import paper_2507_12349_b200 as cos_mod
    cos_mod.load_library()          # fails loudly if libcos_b200.so is missing: there is no fallback
    return cos_mod


def gpu_eval(cos, G, n, n_flavors, lattice, sigmas, all_subsets, ws_limit=None, flags=0, tune=None):
    """G: numpy [n_blocks][d][d][B] -> numpy [n_out][B] through cos_build / cos_eval / cos_free."""
    import torch
    B = G.shape[-1]
    h = cos.cos_build_ex(n, n_flavors, lattice, sigmas, n if all_subsets else 0, flags)
    try:
        if ws_limit is not None:
            cos.cos_set_workspace_limit(h, ws_limit)
        for k, v in (tune or {}).items():
            cos.cos_set_tuning(h, k, v)
        n_out = cos.cos_info(h, "n_out")
        Gd = torch.from_numpy(np.ascontiguousarray(G.reshape(-1, B))).cuda()
        out = torch.full((n_out, B), float("nan"), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, Gd, B, out)
        torch.cuda.synchronize()
        return out.cpu().numpy()
    finally:
        cos.cos_free(h)


def check(got, ref, M, what):
    got, ref, M = np.asarray(got), np.asarray(ref), np.asarray(M)
    assert np.all(np.isfinite(got)), what
    bad = np.abs(got - ref) > TOL * M
    assert not bad.any(), (what, got[bad][:4], ref[bad][:4], M[bad][:4])


def M_lower_bound(G, n, n_sub, nf, uniform, n_assign=4, seed=0):
    """A rigorous LOWER bound of the cancellation scale M (= the sum of |weight| over all connected typed
    contractions, O1 / O3 with absolute=True) that stays cheap at n >= 10: every term of the uniform sum on
    Abar[i][j] = min_lam |A_lam[i][j]| with N_f colours per cycle is dominated by the matching
    SB term, the shift terms (Z nonempty, Eq. 60) are dropped, and of the n_sub^n sublattice assignments
    (Eq. 55) only `n_assign` seeded ones are kept.  Using it in place of M makes the test STRICTER."""
    rng = np.random.default_rng(seed)
    G = np.abs(np.asarray(G))
    assigns = [[0] * n] if n_sub == 1 else [list(rng.integers(0, n_sub, n)) for _ in range(n_assign)]
    assigns = list({tuple(a) for a in assigns})
    total = 0.0
    for a in assigns:
        Abar = oracle.subset_blocks(G, list(range(n)), list(a), n_sub).min(axis=0)
        total += oracle.o3_uniform(Abar, nf, 0.0, False, absolute=True)[0]
    return total


def oracle_vector(G, c, n, n_sub, nf, sigmas, uniform, all_subsets, tier):
    Gc = np.ascontiguousarray(G[..., c])
    ref = oracle.connected_reference(Gc, n, n_sub, nf, sigmas, uniform, all_subsets, tier=tier)
    atier = "o1" if tier == "o1" else "o3"
    M = oracle.connected_reference(Gc, n, n_sub, nf, sigmas, uniform, all_subsets, tier=atier, absolute=True)
    return ref, M


# ------------------------------------------------------------------------------------------------ small orders
@pytest.mark.parametrize("n,nf,all_subsets", [(1, 2, False), (1, 3, True), (2, 2, True), (2, 3, False),
                                              (3, 2, True), (3, 3, True), (4, 2, False), (4, 2, True),
                                              (4, 3, False), (5, 2, False)])
def test_uniform_vs_bruteforce(cos, n, nf, all_subsets):
    """Uniform CoS (Eq. 8-15) against the definition O1 (Eq. 58-63); ragged batch 37."""
    B = 37 if n < 5 else 3
    G = random_matrices(1000 + 10 * n + nf, 1, n, B, scale=0.8)
    got = gpu_eval(cos, G, n, nf, cos.COS_LATTICE_SQUARE, None, all_subsets)
    for c in range(B):
        ref, M = oracle_vector(G, c, n, 1, nf, None, True, all_subsets, "o1")
        check(got[:, c], ref, M, ("uniform", n, nf, c))


@pytest.mark.parametrize("n,nf,all_subsets", [(1, 2, True), (1, 3, False), (2, 2, True), (2, 3, True), (2, 4, False),
                                              (3, 2, True), (3, 3, True), (4, 2, False), (4, 3, True),
                                              (5, 3, False)])
def test_sb_vs_bruteforce(cos, n, nf, all_subsets):
    """SB-CoS with non-uniform shifts (Alg. 3, Eq. 58-72) against the definition O1; Eq. 83 at singletons."""
    B = 33 if n < 4 else (5 if n == 4 else 2)
    rng = np.random.default_rng(50 + n * 7 + nf)
    sig = list(rng.standard_normal(nf) * 0.5)
    G = random_matrices(2000 + 10 * n + nf, nf, n, B, scale=0.8)
    got = gpu_eval(cos, G, n, nf, cos.COS_LATTICE_SQUARE, sig, all_subsets)
    for c in range(B):
        ref, M = oracle_vector(G, c, n, 1, nf, sig, False, all_subsets, "o1")
        check(got[:, c], ref, M, ("sb", n, nf, c))


@pytest.mark.parametrize("n,nf,uniform,all_subsets", [(2, 2, False, True), (3, 2, False, False), (3, 2, True, True),
                                                      (3, 3, False, True), (4, 2, False, False)])
def test_honeycomb_sublattice_sum_vs_bruteforce(cos, n, nf, uniform, all_subsets):
    """Sublattice-summed DAG (Eq. 4, 54-55; n_sub = 2): C = sum over 2^n assignments of O1."""
    B = 9 if n < 4 else 2
    sig = None if uniform else [0.3, -0.3, 0.1][:nf]
    G = random_matrices(3000 + n, 1 if uniform else nf, 2 * n, B, scale=0.7)
    got = gpu_eval(cos, G, n, nf, cos.COS_LATTICE_HONEYCOMB, sig, all_subsets)
    for c in range(B):
        ref, M = oracle_vector(G, c, n, 2, nf, sig, uniform, all_subsets, "o1")
        check(got[:, c], ref, M, ("honeycomb", n, nf, c))


def test_paper_test_vectors(cos):
    """tests/golden/oracle_small.json (written by oracle/ only) + the hand values of SURVEY.md 8(c) TV1-TV4."""
    with open(os.path.join(HERE, "golden", "oracle_small.json")) as f:
        cases = json.load(f)["cases"]
    for case in cases:
        A = np.array(case["A"], dtype=np.float64)
        n = A.shape[-1]
        G = np.ascontiguousarray(np.repeat(A[..., None], 5, axis=-1))
        got = gpu_eval(cos, G, n, case["n_flavors"], cos.COS_LATTICE_SQUARE, case["sigma"], True)
        ref = np.array(case["values_by_bitmask"])
        for c in range(5):
            assert np.allclose(got[:, c], ref, rtol=1e-13, atol=0), (case["name"], got[:, c], ref)


# ------------------------------------------------------------------------------------------------ mid orders
@pytest.mark.parametrize("n", [6, 8, 9])
def test_uniform_all_subsets_vs_determinants(cos, n):
    """n = 6..9, all 2^n - 1 readouts (Eq. 13-15) against the two-determinant CDet route O2a
    (Eq. 53): several tiles and a ragged tail (B = 70)."""
    B = 70
    G = random_matrices(4000 + n, 1, n, B, scale=0.5, diag=-0.45)
    got = gpu_eval(cos, G, n, 2, cos.COS_LATTICE_SQUARE, None, True)
    for c in range(0, B, 5):
        A = np.ascontiguousarray(G[0, :, :, c])
        ref = oracle.o2a_twospin(A, A)
        M = oracle.o3_uniform(A, 2, 0.0, True, absolute=True)
        check(got[:, c], ref, M, ("o2a", n, c))
        check(got[:, c], oracle.o3_uniform(A, 2, 0.0, True), M, ("o3", n, c))


@pytest.mark.parametrize("n,nf", [(6, 3), (7, 2), (6, 4)])
def test_sb_vs_polynomial_and_alg3(cos, n, nf):
    """BASELINE config 4's cross-check: SB-CoS at n <= 7 against the determinant-polynomial route
    (Eq. 34-38) on every subset and the printed Algorithm 3 on the full set."""
    B = 40
    sig = [0.2, 0.0, -0.2, 0.35][:nf]
    G = random_matrices(5000 + n + nf, nf, n, B, scale=0.5, diag=-0.4)
    got = gpu_eval(cos, G, n, nf, cos.COS_LATTICE_SQUARE, sig, True)
    got1 = gpu_eval(cos, G, n, nf, cos.COS_LATTICE_SQUARE, sig, False)
    assert np.array_equal(got[-1], got1[0]) or np.allclose(got[-1], got1[0], rtol=1e-12, atol=0)
    for c in range(0, B, 13):
        A = np.ascontiguousarray(G[..., c])
        ref = oracle.o2b_polynomial(A, sig)
        full = oracle.o3_alg3(A, sig)
        Mfull = oracle.o3_alg3(A, sig, absolute=True)
        check(got[-1, c], full, Mfull, ("alg3", n, nf, c))
        check(got[-1, c], ref[-1], Mfull, ("o2b full", n, nf, c))
        # subsets: bound by the (larger) full-set M is not valid; use each subset's own Alg. 3 bound
        for S in (1, 3, 5, (1 << n) - 2, (1 << (n - 1)) - 1):
            verts = [i for i in range(n) if S >> i & 1]
            As = oracle.subset_blocks(A, verts, [0] * len(verts), 1)
            check(got[S - 1, c], ref[S - 1], oracle.o3_alg3(As, sig, absolute=True), ("o2b subset", S, c))


def test_sb_two_spin_with_shifts_vs_determinants(cos):
    """Two-spin SB-CoS with opposite shifts (config 3's flavour structure, square lattice, n = 8)
    against O2a' (Eq. 49-50, 53)."""
    n, B = 8, 45
    sig = [0.3, -0.3]
    G = random_matrices(6000, 2, n, B, scale=0.5, diag=-0.5)
    got = gpu_eval(cos, G, n, 2, cos.COS_LATTICE_SQUARE, sig, True)
    for c in range(0, B, 11):
        ref = oracle.o2a_twospin(G[0, :, :, c], G[1, :, :, c], sig[0], sig[1])
        for S in (1, 2, 7, 100, 255):
            verts = [i for i in range(n) if S >> i & 1]
            As = oracle.subset_blocks(np.ascontiguousarray(G[..., c]), verts, [0] * len(verts), 1)
            check(got[S - 1, c], ref[S - 1], oracle.o3_alg3(As, sig, absolute=True), ("o2a'", S, c))


def test_honeycomb_n6_vs_determinants(cos):
    """Sublattice-summed two-spin SB DAG at n = 6 (config 3's mode) = sum over 2^6 assignments of O2a'."""
    n, B = 6, 34
    sig = [0.3, -0.3]
    G = random_matrices(6100, 2, 2 * n, B, scale=0.5, diag=-0.5)
    got = gpu_eval(cos, G, n, 2, cos.COS_LATTICE_HONEYCOMB, sig, False)
    for c in (0, 17, 33):
        Gc = np.ascontiguousarray(G[..., c])
        ref = oracle.connected_reference(Gc, n, 2, 2, sig, False, False, tier="o2a")
        M = oracle.connected_reference(Gc, n, 2, 2, sig, False, False, tier="o3", absolute=True)
        check(got[0, c], ref, M, ("honeycomb n6", c))


# ------------------------------------------------------------------------------------------------ edge cases
def test_batch_edge_cases_and_chunking(cos):
    """Empty batch, batch 1, ragged tails, and workspace chunking give identical results (the arithmetic
    per configuration does not depend on the launch shape, so chunked == unchunked bit for bit)."""
    import torch
    n, nf = 5, 2
    G = random_matrices(7000, 1, n, 131, scale=0.6)
    full = gpu_eval(cos, G, n, nf, cos.COS_LATTICE_SQUARE, None, True)
    for B in (1, 31, 32, 33, 64, 131):
        part = gpu_eval(cos, np.ascontiguousarray(G[..., :B]), n, nf, cos.COS_LATTICE_SQUARE, None, True)
        assert np.array_equal(part, full[:, :B]), B
    tiny = gpu_eval(cos, G, n, nf, cos.COS_LATTICE_SQUARE, None, True, ws_limit=1)     # one tile per chunk
    assert np.array_equal(tiny, full)
    h = cos.cos_build(n, nf, cos.COS_LATTICE_SQUARE, None, 0)
    cos.cos_eval(h, torch.empty((n * n, 0), dtype=torch.float64, device="cuda"), 0,
                 torch.empty((1, 0), dtype=torch.float64, device="cuda"))              # no-op
    cos.cos_free(h)
    cos.cos_free(None)


def test_error_paths(cos):
    import torch
    with pytest.raises(cos.CosError):
        cos.cos_build(0, 2, 0, None, 0)
    with pytest.raises(cos.CosError):
        cos.cos_build(13, 2, 0, None, 0)
    with pytest.raises(cos.CosError):
        cos.cos_build(4, 2, 0, None, 3)          # envelope must be 0 or n
    with pytest.raises(cos.CosError):
        cos.cos_build(4, 5, 0, [0.1] * 5, 0)     # SB colours > COS_MAX_COLOURS
    h = cos.cos_build_ex(4, 2, 0, None, 0, flags=cos.COS_BUILD_HOST_ONLY)
    with pytest.raises(cos.CosError):           # host-only handle: no CPU fallback
        cos.cos_eval(h, torch.zeros((16, 4), dtype=torch.float64, device="cuda"), 4,
                     torch.zeros((1, 4), dtype=torch.float64, device="cuda"))
    cos.cos_free(h)


def test_principal_submatrix_property(cos):
    """out[S] must not depend on rows / columns outside S."""
    n, B = 6, 32
    G = random_matrices(7100, 1, n, B, scale=0.6)
    base = gpu_eval(cos, G, n, 3, cos.COS_LATTICE_SQUARE, None, True)
    G2 = G.copy()
    G2[:, 4, :, :] = 17.0
    G2[:, :, 4, :] = -9.0
    pert = gpu_eval(cos, G2, n, 3, cos.COS_LATTICE_SQUARE, None, True)
    for S in range(1, 1 << n):
        if not (S >> 4) & 1:
            assert np.array_equal(base[S - 1], pert[S - 1]), S


# ------------------------------------------------------------------------------------------------ tabulation
@pytest.mark.parametrize("cfg,batch", [(1, 1024), (2, 300), (3, 200), (4, 129), (5, 64)])
def test_tabulation_bit_exact(cos, cfg, batch):
    """Kernel (2) (Eq. 32; readings G17-G18) against oracle.tabulate_reference, bit for bit."""
    import torch
    w = get_config(cfg).scaled(batch=batch)
    table = table_for(w)
    v = draw_vertices(w)
    if cfg == 1:                                  # degenerate cases: equal times and equal sites
        v["tau"][1, :8] = v["tau"][0, :8]
        v["sites"][2, :, :8] = v["sites"][0, :, :8]
        v["tau"][3, 8:12] = 0.0
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    G = torch.empty((w.n_blocks * w.d * w.d, batch), dtype=torch.float64, device="cuda")
    cos.cos_tabulate(tab, w.n, torch.from_numpy(v["sites"]).cuda(), torch.from_numpy(v["tau"]).cuda(), batch, G)
    torch.cuda.synchronize()
    cos.cos_tab_free(tab)
    ref = oracle.tabulate_reference(table, v["sites"], v["tau"])
    assert np.array_equal(G.cpu().numpy(), ref.reshape(-1, batch))


# ------------------------------------------------------------------------------------------------ BASELINE configs
def _tabulated(cos, w):
    import torch
    table = table_for(w)
    v = draw_vertices(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    G = torch.empty((w.n_blocks * w.d * w.d, w.batch), dtype=torch.float64, device="cuda")
    cos.cos_tabulate(tab, w.n, torch.from_numpy(v["sites"]).cuda(), torch.from_numpy(v["tau"]).cuda(), w.batch, G)
    torch.cuda.synchronize()
    cos.cos_tab_free(tab)
    return table, v, G


def _eval_workload(cos, w, G):
    import torch
    h = cos.cos_build(w.n, w.n_flavors, w.lattice, w.sigmas, w.n if w.all_subsets else 0)
    out = torch.full((w.n_out, w.batch), float("nan"), dtype=torch.float64, device="cuda")
    cos.cos_eval(h, G, w.batch, out)
    torch.cuda.synchronize()
    info = cos.dag_summary(h)
    cos.cos_free(h)
    return out.cpu().numpy(), info


def test_config1_full(cos):
    """BASELINE config 1 at full size: every one of the 1024 configurations against O3 (Eq. 8-15) and the
    two-determinant route, a sample against the brute-force definition."""
    w = get_config(1)
    table, v, G = _tabulated(cos, w)
    got, info = _eval_workload(cos, w, G)
    assert (info["n_states"], info["n_edges"], info["n_readout_edges"]) == (191, 522, 13)
    Gh = G.cpu().numpy().reshape(1, w.n, w.n, w.batch)
    for c in range(w.batch):
        A = np.ascontiguousarray(Gh[0, :, :, c])
        M = oracle.o3_uniform(A, 2, 0.0, False, absolute=True)[0]
        check(got[0, c], oracle.o3_uniform(A, 2)[0], M, ("cfg1 o3", c))
        check(got[0, c], oracle.o2a_twospin(A, A)[-1], M, ("cfg1 o2a", c))
        if c % 64 == 0:
            check(got[0, c], oracle.o1_connected(A[None], 2, None, sb=False), M, ("cfg1 o1", c))


def test_config2_full_sampled(cos):
    """BASELINE config 2 at full size (65536 configurations x 255 readouts), sampled configurations
    against O2a on every subset."""
    w = get_config(2)
    table, v, G = _tabulated(cos, w)
    got, info = _eval_workload(cos, w, G)
    assert (info["n_states"], info["n_edges"], info["n_readout_edges"]) == (61353, 313828, 3839)
    assert np.all(np.isfinite(got))
    for c in (0, 1, 31, 32, 4097, 33333, 65535):
        A = np.ascontiguousarray(G[:, c].cpu().numpy().reshape(w.n, w.n))
        M = oracle.o3_uniform(A, 2, 0.0, True, absolute=True)
        check(got[:, c], oracle.o3_uniform(A, 2, 0.0, True), M, ("cfg2 o3", c))
        check(got[:, c], oracle.o2a_twospin(A, A), M, ("cfg2 o2a", c))


def test_config4_full_sampled(cos):
    """BASELINE config 4 at full size (n = 10, three flavours, 8192 configurations), sampled configurations
    against the polynomial route Eq. 34-38 (binary128); bound 1e-10 * (a lower bound of M)."""
    w = get_config(4)
    table, v, G = _tabulated(cos, w)
    got, info = _eval_workload(cos, w, G)
    assert (info["n_states"], info["n_edges"], info["n_readout_edges"]) == (1769937, 16020777, 273)
    assert np.all(np.isfinite(got))
    for c in (0, 33, 8191):
        A = np.ascontiguousarray(G[:, c].cpu().numpy().reshape(3, w.n, w.n))
        ref = oracle.o2b_polynomial(A, w.sigmas)[-1]
        check(got[0, c], ref, M_lower_bound(A, w.n, 1, 3, False), ("cfg4", c))


def _o3_uniform_abs_su2(A):
    return oracle.o3_uniform(A, 2, 0.0, False, absolute=True)[0]


def test_config5_full(cos):
    """BASELINE config 5 at full size (n = 12, 64 configurations): every configuration against O2a (binary128),
    bound 1e-10 M with M from the printed recurrence on |A| (O3 absolute, ~14 s each: run in a process pool)."""
    import multiprocessing as mp
    w = get_config(5)
    table, v, G = _tabulated(cos, w)
    got, info = _eval_workload(cos, w, G)
    assert (info["n_states"], info["n_edges"], info["n_readout_edges"]) == (7280663, 57677458, 133)
    Gh = G.cpu().numpy().reshape(w.n, w.n, w.batch)
    mats = [np.ascontiguousarray(Gh[:, :, c]) for c in range(w.batch)]
    with mp.get_context("fork").Pool(min(16, os.cpu_count() or 1)) as pool:
        Ms = pool.map(_o3_uniform_abs_su2, mats, chunksize=1)
    for c in range(w.batch):
        ref = oracle.o2a_twospin(mats[c], mats[c])[-1]
        check(got[0, c], ref, Ms[c], ("cfg5", c))


def test_config3_full_sampled(cos):
    """BASELINE config 3 at full size (honeycomb, two spins, opposite shifts, n = 10, 3.9e7 states, 16384 configurations;
    the 64 GiB workspace budget makes cos_eval walk the batch in chunks of 17 tiles, as in bench.py); sampled
    configurations against the sum over 2^10 sublattice assignments of O2a' (binary128)."""
    w = get_config(3)
    table, v, G = _tabulated(cos, w)
    got, info = _eval_workload(cos, w, G)
    assert (info["n_states"], info["n_edges"], info["n_readout_edges"]) == (39320580, 422359128, 688)
    assert np.all(np.isfinite(got))
    for c in (0, 8191, 16383):
        Gc = np.ascontiguousarray(G[:, c].cpu().numpy().reshape(2, w.d, w.d))
        ref = oracle.connected_reference(Gc, w.n, 2, 2, w.sigmas, False, False, tier="o2a")[0]
        check(got[0, c], ref, M_lower_bound(Gc, w.n, 2, 2, False, n_assign=4, seed=c), ("cfg3", c))


@pytest.mark.parametrize("n,nf,lattice,sb,all_subsets", [(4, 2, 0, False, False), (5, 3, 0, True, True),
                                                          (3, 2, 1, True, True), (6, 3, 0, True, False)])
def test_fused_and_layered_paths_agree(cos, n, nf, lattice, sb, all_subsets):
    """Small DAGs run in ONE launch (cos_fused_kernel); COS_BUILD_NO_FUSED / cos_set_tuning("fused", 0) force the
    per-layer kernels.  Both walk the same program with the same arithmetic order, so the outputs must be bit-identical
    (and equal the oracle, tested above).  The launch tuning knobs must not change a bit either."""
    n_sub = 2 if lattice else 1
    sig = [0.3, -0.2, 0.1][:nf] if sb else None
    G = random_matrices(50 + n, nf if sb else 1, n * n_sub, 77, scale=0.5)
    a = gpu_eval(cos, G, n, nf, lattice, sig, all_subsets)
    a_chunked = gpu_eval(cos, G, n, nf, lattice, sig, all_subsets, ws_limit=1)      # one tile per chunk
    b = gpu_eval(cos, G, n, nf, lattice, sig, all_subsets, flags=cos.COS_BUILD_NO_FUSED)
    b2 = gpu_eval(cos, G, n, nf, lattice, sig, all_subsets, tune={"fused": 0, "pdl": 0, "prefetch": 0, "warps_per_cta": 4,
                                                                   "blocks_per_cta_cap": 3, "tiles_per_chunk": 2})
    assert np.all(np.isfinite(a))
    assert np.array_equal(a, b) and np.array_equal(a, a_chunked) and np.array_equal(a, b2)


def test_fused_flag_is_reported(cos):
    h = cos.cos_build(4, 2, cos.COS_LATTICE_SQUARE, None, 0)
    h2 = cos.cos_build_ex(4, 2, cos.COS_LATTICE_SQUARE, None, 0, cos.COS_BUILD_NO_FUSED)
    h3 = cos.cos_build(8, 2, cos.COS_LATTICE_SQUARE, None, 0)       # too large for the fused kernel
    try:
        assert cos.cos_info(h, "fused") == 1 and cos.cos_info(h2, "fused") == 0 and cos.cos_info(h3, "fused") == 0
        cos.cos_set_tuning(h3, "fused", 1)                           # ignored: the DAG does not qualify
        assert cos.cos_info(h3, "fused") == 0
        with pytest.raises(cos.CosError) as ei:
            cos.cos_set_tuning(h, "warps_per_cta", 17)
        assert ei.value.code == cos.COS_EINVAL
        with pytest.raises(cos.CosError):
            cos.cos_set_tuning(h, 99, 1)
    finally:
        cos.cos_free(h); cos.cos_free(h2); cos.cos_free(h3)


def test_four_flavours_per_layer_kernels(cos):
    """N_f = 4 (the largest colour count the state carries) at n = 7 -- beyond the fused small-DAG path -- against the
    polynomial route Eq. 34-38 generalised to any N_f (reading G13) and against Algorithm 3 as printed."""
    n, nf, B = 7, 4, 40
    sig = [0.25, -0.1, 0.0, 0.3]
    G = random_matrices(404, nf, n, B, scale=0.45, diag=-0.4)
    got = gpu_eval(cos, G, n, nf, cos.COS_LATTICE_SQUARE, sig, False)
    for c in (0, 17, 39):
        A = np.ascontiguousarray(G[..., c])
        M = oracle.o3_alg3(A, sig, absolute=True)
        check(got[0, c], oracle.o2b_polynomial(A, sig)[-1], M, ("nf4 o2b", c))
        check(got[0, c], oracle.o3_alg3(A, sig), M, ("nf4 o3", c))


def test_honeycomb_uniform_long_rows(cos):
    """Uniform CoS with the sublattice sum (Algorithm 2; Eq. 4, 55) at n = 7: d = 14 endpoints, rows of up
    to 14 states (the MAXL = 20 kernels without shifts), against the sum over 2^7 assignments of the two-determinant
    route."""
    n, B = 7, 36
    G = random_matrices(505, 1, 2 * n, B, scale=0.4, diag=-0.45)
    got = gpu_eval(cos, G, n, 2, cos.COS_LATTICE_HONEYCOMB, None, False)
    for c in (0, 35):
        Gc = np.ascontiguousarray(G[..., c])
        ref = oracle.connected_reference(Gc, n, 2, 2, None, True, False, tier="o2a")
        M = oracle.connected_reference(Gc, n, 2, 2, None, True, False, tier="o3", absolute=True)
        check(got[:, c], ref, M, ("honeycomb uniform", c))
