"""GPU parity of the determinant-polynomial route (cos_det_eval; Eq. 34-38) against the CPU
oracle, element by element, and against the DAG path (cos_eval) on the same inputs.  Needs a B200 (`-m gpu`).

Acceptance bound: |GPU - oracle| <= tol * R, R = the route's own absolute-value evaluation (oracle O2b with
absolute=2: permanents of |A| for the minors, |sigma|, every minus sign of Eq. 38 turned into a plus).  R is larger
than the DAG's M (it also contains the disconnected products that Eq. 38 subtracts) and is what bounds the rounding
error of THIS route (include/cos.h, cos_det_eval); tol = 1e6 x the unit roundoff of the working precision:
1e-10 in fp64 (north_star's figure), 1e-26 in double-double.  The oracle computes in binary128 (~1e-34).
"""
import numpy as np
import pytest

import oracle
from cos_workloads import draw_vertices, get_config, random_matrices
from cos_workloads.tables import table_for

pytestmark = pytest.mark.gpu

TOL = {0: 1e-10, 1: 1e-26}          # COS_DET_FP64, COS_DET_DD
PRECISIONS = [0, 1]


@pytest.fixture(scope="module")
def cos():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    torch.cuda.set_device(0)
    import paper_2507_12349_b200 as cos_mod
    cos_mod.load_library()
    return cos_mod


def det_eval(cos, G, n, nf, sigmas, prec=0, lattice=0):
    """G: numpy [n_blocks][d][d][B] -> numpy [2^n-1][B] through cos_det_eval."""
    import torch
    B = G.shape[-1]
    nb = G.shape[0]
    Gd = torch.from_numpy(np.ascontiguousarray(G.reshape(-1, B))).cuda()
    out = torch.full(((1 << n) - 1, B), float("nan"), dtype=torch.float64, device="cuda")
    nbytes = cos.cos_det_workspace_bytes(n, nb, prec, B)
    assert nbytes > 0
    work = torch.empty((nbytes + 7) // 8, dtype=torch.float64, device="cuda")
    cos.cos_det_eval(n, nf, nb, sigmas, prec, Gd, B, out, work, lattice=lattice)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def dag_eval(cos, G, n, nf, sigmas, lattice=0):
    import torch
    B = G.shape[-1]
    h = cos.cos_build(n, nf, lattice, sigmas, n)
    try:
        Gd = torch.from_numpy(np.ascontiguousarray(G.reshape(-1, B))).cuda()
        out = torch.full(((1 << n) - 1, B), float("nan"), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, Gd, B, out)
        torch.cuda.synchronize()
        return out.cpu().numpy()
    finally:
        cos.cos_free(h)


def check(got, ref, M, what, tol=1e-10):
    """|got - ref| <= tol * M, plus half an ulp of the fp64 output (the double-double result is rounded to fp64)."""
    got, ref, M = np.asarray(got), np.asarray(ref), np.asarray(M)
    assert np.all(np.isfinite(got)), what
    bad = np.abs(got - ref) > tol * M + 2.3e-16 * np.abs(ref)
    assert not bad.any(), (what, got[bad][:4], ref[bad][:4], M[bad][:4])


@pytest.mark.parametrize("prec", PRECISIONS)
@pytest.mark.parametrize("n,nf", [(1, 2), (1, 3), (2, 2), (2, 3), (3, 2), (3, 3), (4, 3), (5, 2)])
def test_det_route_vs_bruteforce(cos, n, nf, prec):
    """Every subset value against the definition Eq. 58-63 (brute-force Wick sum O1 in fp64, convention Eq. 83),
    non-uniform matrices and shifts; B = 37 is one full tile and a ragged one.  O1 is an fp64 sum, so the bound is
    the fp64 one for both precisions."""
    B = 37
    sig = [0.5, -1.0 / 3.0, 0.25][:nf]
    G = random_matrices(9100 + 10 * n + nf, nf, n, B, scale=0.8)
    got = det_eval(cos, G, n, nf, sig, prec)
    for c in range(0, B, 6 if n < 5 else 18):
        A = np.ascontiguousarray(G[..., c])
        ref = oracle.o1_all_subsets(A, nf, sig, sb=True)
        R = oracle.o2b_polynomial(A, sig, absolute=2)
        check(got[:, c], ref, R, ("o1", n, nf, c), TOL[0])


@pytest.mark.parametrize("prec", PRECISIONS)
def test_det_route_paper_test_vectors(cos, prec):
    """SURVEY.md 8(c) TV3 / TV4 (exact rationals; brute force, Alg. 3 and Eq. 34-38 agree on them)."""
    A0, A1, A2 = [[1, 2], [3, 4]], [[2, -1], [1, 3]], [[-1, 1], [2, 1]]
    G = np.array([A0, A1], dtype=np.float64)[..., None].repeat(3, axis=-1)
    got = det_eval(cos, G, 2, 2, [0.5, -1.0 / 3.0], prec)
    assert np.allclose(got[:, 1], [11.0 / 3.0, 26.0, -2018.0 / 9.0], rtol=1e-13, atol=0)
    G = np.array([A0, A1, A2], dtype=np.float64)[..., None].repeat(2, axis=-1)
    got = det_eval(cos, G, 2, 3, [0.5, 0.0, -0.5], prec)
    assert np.allclose(got[:, 0], [0.0, 41.0, -276.0], rtol=1e-13, atol=1e-13)


@pytest.mark.parametrize("prec", PRECISIONS)
@pytest.mark.parametrize("n,nf", [(6, 3), (7, 3), (8, 2), (9, 2)])
def test_det_route_vs_polynomial_oracle(cos, n, nf, prec):
    """Against the oracle's own Eq. 34-38 in binary128 on every subset; several tiles and a ragged tail."""
    B = 70
    sig = [0.2, 0.0, -0.2][:nf] if nf == 3 else [0.3, -0.3]
    G = random_matrices(9200 + 10 * n + nf, nf, n, B, scale=0.5, diag=-0.45)
    got = det_eval(cos, G, n, nf, sig, prec)
    for c in range(0, B, 23):
        A = np.ascontiguousarray(G[..., c])
        check(got[:, c], oracle.o2b_polynomial(A, sig), oracle.o2b_polynomial(A, sig, absolute=2), ("o2b", n, nf, c), TOL[prec])


@pytest.mark.parametrize("prec", PRECISIONS)
@pytest.mark.parametrize("n,nf", [(5, 2), (5, 3), (8, 2)])
def test_det_route_uniform_blocks(cos, n, nf, prec):
    """n_blocks = 1, no shifts: every flavour reads block 0 (Eq. 33) and the result is the uniform CoS value with loop
    factor N_f -- the uniform recurrence Eq. 8-15 (O3, fp64) and, for two spins, det^2 + CDet (O2a,
    binary128)."""
    B = 33
    G = random_matrices(9300 + n + nf, 1, n, B, scale=0.6, diag=-0.4)
    got = det_eval(cos, G, n, nf, None, prec)
    for c in (0, 16, 32):
        A = np.ascontiguousarray(G[0, :, :, c])
        R = oracle.o2b_polynomial(np.stack([A] * nf), [0.0] * nf, absolute=2)
        check(got[:, c], oracle.o3_uniform(A, nf, 0.0, True), R, ("o3 uniform", n, nf, c), TOL[0])
        if nf == 2:
            check(got[:, c], oracle.o2a_twospin(A, A), R, ("o2a", n, c), TOL[prec])


def _tabulated(cos, w):
    import torch
    table = table_for(w)
    v = draw_vertices(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    try:
        G = torch.empty((w.n_blocks * w.d * w.d, w.batch), dtype=torch.float64, device="cuda")
        cos.cos_tabulate(tab, w.n, torch.from_numpy(v["sites"]).cuda(), torch.from_numpy(v["tau"]).cuda(), w.batch, G)
        torch.cuda.synchronize()
    finally:
        cos.cos_tab_free(tab)
    return G


@pytest.mark.parametrize("prec", PRECISIONS)
@pytest.mark.parametrize("cfg,n,nf", [(4, 6, 3), (4, 8, 3), (2, 8, 2)])
def test_det_route_and_dag_on_tabulated_propagators(cos, cfg, n, nf, prec):
    """The two GPU evaluators on the same tabulated propagators (config-4- and config-2-shaped inputs at reduced order):
    DAG with all-subset readouts (Eq. 13-15) vs minors + Eq. 38.  On physical propagators the connected value is many
    orders below the moments (R / |C| up to ~1e17 at n = 8), so the fp64 route is only held to ITS bound 1e-10 R, while
    the double-double route must reproduce the binary128 oracle to fp64 accuracy and therefore the DAG within the
    DAG's own bound 1e-10 M on EVERY subset of EVERY configuration."""
    w = get_config(cfg).scaled(batch=129, n=n)
    G = _tabulated(cos, w)
    Gn = G.cpu().numpy().reshape(w.n_blocks, n, n, w.batch)
    sb = w.alphas is not None
    sig = list(w.sigmas) if sb else None
    got_det = det_eval(cos, Gn, n, nf, sig, prec)
    got_dag = dag_eval(cos, Gn, n, nf, sig)
    for c in (0, 64, 128):
        A = np.ascontiguousarray(Gn[..., c])
        Af = A if sb else np.stack([A[0]] * nf)
        sg = sig if sb else [0.0] * nf
        ref = oracle.o2b_polynomial(Af, sg)
        check(got_det[:, c], ref, oracle.o2b_polynomial(Af, sg, absolute=2), ("det", cfg, n, c), TOL[prec])
        check(got_dag[:, c], ref, oracle.o2b_polynomial(Af, sg, absolute=True), ("dag", cfg, n, c), 1e-10)
    if prec == 1:
        # every configuration, route against route: |C_S| / M >= 1e-4 on these inputs (typically 0.03-0.7),
        # so 1e-10 M <= 1e-6 |C|; the two routes agree to ~1e-13 relative
        rel = np.abs(got_det - got_dag) / np.abs(got_dag)
        assert np.max(rel) <= 1e-9, np.max(rel)


def test_det_route_config4_full(cos):
    """BASELINE config 4 at full size (n = 10, three flavours, 8192 configurations): the determinant route in
    double-double on the device against the DAG's full-order output on EVERY configuration (the on-device cross-check of
    SURVEY 8(f).3), and against the binary128 oracle on sampled configurations (all 1023 subsets)."""
    import torch
    w = get_config(4)
    n = w.n
    G = _tabulated(cos, w)
    out = torch.full(((1 << n) - 1, w.batch), float("nan"), dtype=torch.float64, device="cuda")
    work = torch.empty((cos.cos_det_workspace_bytes(n, 3, cos.COS_DET_DD, w.batch) + 7) // 8, dtype=torch.float64,
                       device="cuda")
    cos.cos_det_eval(n, 3, 3, w.sigmas, cos.COS_DET_DD, G, w.batch, out, work)
    h = cos.cos_build(n, 3, cos.COS_LATTICE_SQUARE, w.sigmas, 0)
    try:
        dag = torch.empty((1, w.batch), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, G, w.batch, dag)
        torch.cuda.synchronize()
    finally:
        cos.cos_free(h)
    det_full = out[-1].cpu().numpy()
    dag_full = dag[0].cpu().numpy()
    assert np.all(np.isfinite(det_full))
    for c in (0, 8191):
        A = np.ascontiguousarray(G[:, c].cpu().numpy().reshape(3, n, n))
        ref = oracle.o2b_polynomial(A, w.sigmas)
        check(out[:, c].cpu().numpy(), ref, oracle.o2b_polynomial(A, w.sigmas, absolute=2), ("cfg4 det", c), TOL[1])
    # R / |C| ~ 1e22 at n = 10: double-double (1e-32) leaves ~1e-10 relative on the full-order value, binary128 ~1e-12
    rel = np.abs(det_full - dag_full) / np.abs(dag_full)
    assert np.median(rel) <= 1e-9 and np.max(rel) <= 1e-5, (np.median(rel), np.max(rel))


# ------------------------------------------------------------------------------------------------ honeycomb (Eq. 54-55)
@pytest.mark.parametrize("prec", PRECISIONS)
@pytest.mark.parametrize("n,nf", [(1, 2), (2, 2), (2, 3), (3, 2), (3, 3), (4, 2)])
def test_det_route_honeycomb_vs_bruteforce(cos, n, nf, prec):
    """Sublattice-summed route (moments summed over the 2^|T| labels before Eq. 38) against the sum over assignments of
    the brute-force connected sums O1 (Eq. 55), every subset; scale R = sum over assignments of the route's scale."""
    B = 9 if n < 4 else 3
    sig = [0.3, -0.3, 0.1][:nf]
    G = random_matrices(9500 + 10 * n + nf, nf, 2 * n, B, scale=0.7)
    got = det_eval(cos, G, n, nf, sig, prec, lattice=cos.COS_LATTICE_HONEYCOMB)
    for c in range(B):
        Gc = np.ascontiguousarray(G[..., c])
        ref = oracle.connected_reference(Gc, n, 2, nf, sig, False, True, tier="o1")
        R = oracle.connected_reference(Gc, n, 2, nf, sig, False, True, tier="o2b", absolute=2)
        check(got[:, c], ref, R, ("honeycomb o1", n, nf, c), TOL[0])


@pytest.mark.parametrize("prec", PRECISIONS)
@pytest.mark.parametrize("n", [5, 6])
def test_det_route_honeycomb_config3_shape_vs_dag(cos, n, prec):
    """Config-3-shaped inputs (honeycomb, two spins, opposite shifts, tabulated 2x2 sublattice blocks) at reduced order:
    the sublattice-summed determinant route vs the oracle (sum over assignments of O2b in binary128) on sampled
    configurations, and in double-double vs the honeycomb DAG with all-subset readouts on every configuration."""
    w = get_config(3).scaled(batch=65, n=n)
    G = _tabulated(cos, w)
    Gn = G.cpu().numpy().reshape(w.n_blocks, 2 * n, 2 * n, w.batch)
    sig = list(w.sigmas)
    got_det = det_eval(cos, Gn, n, 2, sig, prec, lattice=cos.COS_LATTICE_HONEYCOMB)
    got_dag = dag_eval(cos, Gn, n, 2, sig, lattice=cos.COS_LATTICE_HONEYCOMB)
    for c in (0, 64):
        Gc = np.ascontiguousarray(Gn[..., c])
        ref = oracle.connected_reference(Gc, n, 2, 2, sig, False, True, tier="o2b")
        R = oracle.connected_reference(Gc, n, 2, 2, sig, False, True, tier="o2b", absolute=2)
        M = oracle.connected_reference(Gc, n, 2, 2, sig, False, True, tier="o2b", absolute=True)
        # the reference adds the 2^|T| per-assignment values in fp64, so it is itself only good to ~1e-16 M: the fp64 route
        # is held to its own bound 1e-10 R, the double-double route to the DAG's (much smaller) 1e-10 M
        check(got_det[:, c], ref, R if prec == 0 else M, ("honeycomb det", n, c), 1e-10)
        check(got_dag[:, c], ref, M, ("honeycomb dag", n, c), 1e-10)
    if prec == 1:
        rel = np.abs(got_det - got_dag) / np.abs(got_dag)
        assert np.max(rel) <= 1e-9, np.max(rel)


def test_det_route_honeycomb_config3_n10_sampled(cos):
    """BASELINE config 3 at its order (n = 10, honeycomb, 4.2e8-edge DAG) on its first 128 configurations: the
    double-double sublattice-summed determinant route (1024 assignments) against the DAG's output on every one of them,
    and against the oracle (sum over assignments of the two-determinant route O2a', binary128) on one."""
    import torch
    w = get_config(3).scaled(batch=128)
    n = w.n
    G = _tabulated(cos, w)
    out = torch.full(((1 << n) - 1, w.batch), float("nan"), dtype=torch.float64, device="cuda")
    work = torch.empty((cos.cos_det_workspace_bytes(n, 2, cos.COS_DET_DD, w.batch) + 7) // 8, dtype=torch.float64,
                       device="cuda")
    cos.cos_det_eval(n, 2, 2, w.sigmas, cos.COS_DET_DD, G, w.batch, out, work, lattice=cos.COS_LATTICE_HONEYCOMB)
    h = cos.cos_build(n, 2, cos.COS_LATTICE_HONEYCOMB, w.sigmas, 0)
    try:
        dag = torch.empty((1, w.batch), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, G, w.batch, dag)
        torch.cuda.synchronize()
    finally:
        cos.cos_free(h)
    det_full, dag_full = out[-1].cpu().numpy(), dag[0].cpu().numpy()
    assert np.all(np.isfinite(det_full))
    rel = np.abs(det_full - dag_full) / np.abs(dag_full)
    assert np.median(rel) <= 1e-8 and np.max(rel) <= 1e-4, (np.median(rel), np.max(rel))
    Gc = np.ascontiguousarray(G[:, 5].cpu().numpy().reshape(2, 2 * n, 2 * n))
    ref = oracle.connected_reference(Gc, n, 2, 2, w.sigmas, False, False, tier="o2a")[0]
    assert abs(det_full[5] - ref) <= 1e-6 * abs(ref) and abs(dag_full[5] - ref) <= 1e-6 * abs(ref), (det_full[5], dag_full[5], ref)


def _dag_full(cos, w, G):
    import torch
    h = cos.cos_build(w.n, w.n_flavors, w.lattice, w.sigmas, w.n if w.all_subsets else 0)
    try:
        out = torch.empty((w.n_out, w.batch), dtype=torch.float64, device="cuda")
        cos.cos_eval(h, G, w.batch, out)
        torch.cuda.synchronize()
        return out
    finally:
        cos.cos_free(h)


def test_det_route_config2_full_every_output(cos):
    """BASELINE config 2 at full size (n = 8, two spins, 65,536 configurations x 255 readouts): every output of the DAG
    against the double-double determinant route (one flavour-uniform block, no shifts: H(T) = 2^|T| det(A[T])^2)."""
    import torch
    w = get_config(2)
    G = _tabulated(cos, w)
    dag = _dag_full(cos, w, G)
    det = torch.empty_like(dag)
    work = torch.empty((cos.cos_det_workspace_bytes(w.n, 1, cos.COS_DET_DD, w.batch) + 7) // 8, dtype=torch.float64,
                       device="cuda")
    cos.cos_det_eval(w.n, 2, 1, None, cos.COS_DET_DD, G, w.batch, det, work)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(det).all())
    rel = ((det - dag).abs() / dag.abs()).cpu().numpy()
    # the DAG's fp64 error is ~1e-15 M (the route's, in double-double, is far below), so the relative difference is
    # ~1e-15 M / |C_S|: among 1.7e7 outputs a few cancel to |C_S| / M ~ 1e-9 (the element-wise 1e-10 M bound is checked
    # against the oracle on sampled configurations in test_gpu_parity.py::test_config2_full_sampled)
    assert np.median(rel) <= 1e-13 and np.quantile(rel, 0.9999) <= 1e-10 and np.max(rel) <= 1e-5, \
        (np.median(rel), np.quantile(rel, 0.9999), np.max(rel))
    A = np.ascontiguousarray(G[:, 77].cpu().numpy().reshape(w.n, w.n))
    ref = oracle.o2a_twospin(A, A)
    check(det[:, 77].cpu().numpy(), ref, oracle.o2b_polynomial(np.stack([A, A]), [0.0, 0.0], absolute=2), "cfg2 det", TOL[1])


def test_det_route_config5_precision_limit(cos):
    """BASELINE config 5 (n = 12, beta = 8, 64 configurations): where the determinant route stops being a cross-check.
    The connected value is ~1e-27 of the route's scale R here, so even double-double (~1e-32 per operation) keeps only
    ~5 digits (median) -- the reason the paper's determinant route needs extended precision and the DAG,
    whose error scales with the connected M, does not.  Gross agreement only; the DAG itself is checked against the
    binary128 oracle in test_gpu_parity.py::test_config5_full."""
    import torch
    w = get_config(5)
    G = _tabulated(cos, w)
    dag = _dag_full(cos, w, G)[0].cpu().numpy()
    out = torch.empty(((1 << w.n) - 1, w.batch), dtype=torch.float64, device="cuda")
    work = torch.empty((cos.cos_det_workspace_bytes(w.n, 1, cos.COS_DET_DD, w.batch) + 7) // 8, dtype=torch.float64,
                       device="cuda")
    cos.cos_det_eval(w.n, 2, 1, None, cos.COS_DET_DD, G, w.batch, out, work)
    torch.cuda.synchronize()
    det = out[-1].cpu().numpy()
    assert np.all(np.isfinite(det))
    rel = np.abs(det - dag) / np.abs(dag)
    assert np.median(rel) <= 1e-3, (np.median(rel), np.max(rel))
    # the lower orders of the same call are resolved: every subset of size <= 8 of configuration 9 against O2a (binary128)
    A = np.ascontiguousarray(G[:, 9].cpu().numpy().reshape(w.n, w.n))
    ref = oracle.o2a_twospin(A, A)
    got = out[:, 9].cpu().numpy()
    small = np.array([bin(T).count("1") <= 8 for T in range(1, 1 << w.n)])
    assert np.max(np.abs(got[small] - ref[small]) / np.abs(ref[small])) <= 1e-6


def test_det_route_edge_cases_and_errors(cos):
    import torch
    n, nf = 3, 3
    G = random_matrices(9400, nf, n, 1, scale=0.7)
    A = np.ascontiguousarray(G[..., 0])
    for prec in PRECISIONS:
        got = det_eval(cos, G, n, nf, [0.1, 0.2, 0.3], prec)                    # batch = 1
        check(got[:, 0], oracle.o1_all_subsets(A, nf, [0.1, 0.2, 0.3], sb=True),
              oracle.o2b_polynomial(A, [0.1, 0.2, 0.3], absolute=2), "batch 1")
    Gd = torch.zeros((nf * n * n, 4), dtype=torch.float64, device="cuda")
    out = torch.full((7, 4), 5.0, dtype=torch.float64, device="cuda")
    work = torch.empty(cos.cos_det_workspace_bytes(n, nf, 1, 4) // 8 + 1, dtype=torch.float64, device="cuda")
    cos.cos_det_eval(n, nf, nf, None, 0, Gd, 0, out, work)               # batch = 0: no-op
    torch.cuda.synchronize()
    assert float(out.min()) == 5.0
    for prec in PRECISIONS:
        out.fill_(5.0)
        cos.cos_det_eval(n, nf, nf, None, prec, Gd, 4, out, work)        # singular everywhere: all minors 0 -> all zeros
        torch.cuda.synchronize()
        assert float(out.abs().max()) == 0.0
    assert cos.cos_det_workspace_bytes(0, 1, 0, 4) == -1 and cos.cos_det_workspace_bytes(13, 1, 0, 4) == -1
    assert cos.cos_det_workspace_bytes(3, 1, 2, 4) == -1
    assert cos.cos_det_workspace_bytes(3, 3, 1, 4) > cos.cos_det_workspace_bytes(3, 3, 0, 4) > 0
    with pytest.raises(cos.CosError) as e:
        cos.cos_det_eval(n, 3, 3, None, 0, Gd, 4, out, work, lattice=2)
    assert e.value.code == cos.COS_EINVAL
    Gd4 = torch.zeros((4 * n * n, 4), dtype=torch.float64, device="cuda")     # the binding checks tensor sizes first
    for args, code in (((n, 4, 4, None, 0, Gd4, 4, out, work), cos.COS_EUNSUPPORTED),
                       ((n, 3, 2, None, 0, Gd, 4, out, work), cos.COS_EINVAL),
                       ((n, 3, 3, None, 7, Gd, 4, out, work), cos.COS_EINVAL),
                       ((n, 3, 3, None, 1, Gd, 4, out, work[:8]), cos.COS_EINVAL),
                       ((n, 3, 3, None, 1, Gd, 4, out, work.view(torch.uint8)[8:]), cos.COS_EINVAL)):
        with pytest.raises(cos.CosError) as e:
            cos.cos_det_eval(*args)
        assert e.value.code == code
