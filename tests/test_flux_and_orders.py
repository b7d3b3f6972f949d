"""Many-configuration weights (Eq. 6-7) and partial readout sets (allowed orders U; requested-output
pruning Eq. 21-24): oracle pins and host-compiler structure on CPU, CUDA parity with -m gpu."""
import math

import numpy as np
import pytest

import oracle
from cos_workloads import random_matrices


# ---------------------------------------------------------------------------------------- oracle pins (CPU)
def test_flux_hand_value_n2():
    """N = 2 written out by hand from Eq. 6-7: subsets {0}, {1} (order 1, binom 2) and {0,1} (order 2, binom 1)."""
    C = np.array([2.0, -3.0, 5.0])           # C_{0}, C_{1}, C_{01}
    Q = np.array([0.5, 0.25, 2.0])
    lam = [0.0, 4.0, -1.5]
    W, phi = oracle.flux_weights(C, Q, lam)
    assert np.array_equal(phi, np.array([4.0, -3.0, -15.0]))
    assert W == 4.0 / 2 + 3.0 / 2 + 15.0 / 1
    W1, phi1 = oracle.flux_weights(C, Q, lam, order_mask=1 << 2)          # U = {2}
    assert W1 == 15.0 and np.array_equal(phi1, np.array([0.0, 0.0, -15.0]))
    W2, _ = oracle.flux_weights(C, None, lam, order_mask=1 << 1)          # U = {1}, Q = 1
    assert W2 == 8.0 / 2 + 12.0 / 2


def test_flux_invariants():
    """Equal |Phi| on every subset of one order contributes |Phi| once (the binom normalisation of Eq. 7);
    W is invariant under relabelling the vertices and homogeneous of degree one in lambda."""
    N = 5
    rng = np.random.default_rng(3)
    orders = np.array([bin(S).count("1") for S in range(1, 1 << N)])
    lam = rng.standard_normal(N + 1)
    C = np.ones((1 << N) - 1)
    W, _ = oracle.flux_weights(C, None, lam)
    assert abs(W - np.abs(lam[1:]).sum()) < 1e-14
    C = rng.standard_normal((1 << N) - 1)
    Q = rng.random((1 << N) - 1)
    W, phi = oracle.flux_weights(C, Q, lam)
    perm = rng.permutation(N)
    def relabel(S):
        return sum(1 << int(perm[i]) for i in range(N) if S >> i & 1)
    Cp, Qp = np.zeros_like(C), np.zeros_like(Q)
    for S in range(1, 1 << N):
        Cp[relabel(S) - 1], Qp[relabel(S) - 1] = C[S - 1], Q[S - 1]
    Wp, _ = oracle.flux_weights(Cp, Qp, lam)
    assert abs(W - Wp) <= 1e-13 * W
    W3, _ = oracle.flux_weights(C, Q, -3.0 * lam)
    assert abs(W3 - 3.0 * W) <= 1e-13 * W
    direct = sum(abs(lam[orders[i]] * C[i] * Q[i]) / math.comb(N, orders[i]) for i in range(len(C)))
    assert abs(W - direct) <= 1e-13 * W


# ---------------------------------------------------------------------------------------- host compiler (CPU)
@pytest.fixture(scope="module")
def cos():
    from paper_2507_12349_b200 import build as b
    b.build()
    import paper_2507_12349_b200 as cos_mod
    cos_mod.load_library()
    return cos_mod


def _summary(cos, n, nf, lat, sh, mask):
    h = cos.cos_build_orders(n, nf, lat, sh, mask, flags=cos.COS_BUILD_HOST_ONLY)
    try:
        return cos.dag_summary(h)
    finally:
        cos.cos_free(h)


def test_partial_orders_prune_the_dag(cos):
    """Requesting fewer orders keeps fewer states (K_l = F_l ^ B_l, Eq. 23): every order = the all-subset DAG,
    only the top order = the single-output DAG, and the pruning pass really removes forward-reachable states."""
    n = 6
    h = cos.cos_build_ex(n, 2, 0, None, n, flags=cos.COS_BUILD_HOST_ONLY)
    full = cos.dag_summary(h); cos.cos_free(h)
    h = cos.cos_build_ex(n, 2, 0, None, 0, flags=cos.COS_BUILD_HOST_ONLY)
    single = cos.dag_summary(h); cos.cos_free(h)
    every = _summary(cos, n, 2, 0, None, (2 << n) - 2)
    top = _summary(cos, n, 2, 0, None, 1 << n)
    low = _summary(cos, n, 2, 0, None, (1 << 1) | (1 << 2))
    mid = _summary(cos, n, 2, 0, None, 1 << 3)
    assert every["n_states"] == full["n_states"] and every["n_edges"] == full["n_edges"]
    assert top["n_states"] == single["n_states"] and top["n_edges"] == single["n_edges"]
    assert top["n_readout_edges"] == single["n_readout_edges"] and top["n_out"] == 2 ** n - 1
    assert low["n_states"] < mid["n_states"] < full["n_states"]
    assert low["n_states_unpruned"] > low["n_states"]          # states beyond layer 3 are reachable but unproductive
    assert sum(low["layer_states"][4:]) == 0                   # l(S) = 2|S| - 1 <= 3 (Eq. 13)
    assert low["order_mask"] == 6 and full["order_mask"] == (2 << n) - 2 and single["order_mask"] == 0
    with pytest.raises(cos.CosError):
        cos.cos_build_orders(n, 2, 0, None, 1 << (n + 1), flags=cos.COS_BUILD_HOST_ONLY)
    with pytest.raises(cos.CosError):
        cos.cos_build_orders(n, 2, 0, None, 1, flags=cos.COS_BUILD_HOST_ONLY)


# ---------------------------------------------------------------------------------------- CUDA parity (GPU)
@pytest.mark.gpu
@pytest.mark.parametrize("n,nf,sb,mask", [(4, 2, False, (1 << 2) | (1 << 4)), (4, 3, True, 1 << 3), (5, 2, False, 1 << 1),
                                          (3, 3, True, (1 << 1) | (1 << 3)), (4, 2, True, 1 << 4)])
def test_partial_orders_vs_bruteforce(cos, n, nf, sb, mask):
    """Requested subsets equal the definition O1 (Eq. 58-63) on the principal sub-blocks; the others are zero."""
    import torch
    B = 45
    sig = [0.3, -0.2, 0.1][:nf] if sb else None
    G = random_matrices(11 + n, nf if sb else 1, n, B, scale=0.6)
    h = cos.cos_build_orders(n, nf, 0, sig, mask)
    out = torch.full(((1 << n) - 1, B), float("nan"), dtype=torch.float64, device="cuda")
    cos.cos_eval(h, torch.from_numpy(G.reshape(-1, B)).cuda(), B, out)
    torch.cuda.synchronize()
    cos.cos_free(h)
    got = out.cpu().numpy()
    orders = np.array([bin(S).count("1") for S in range(1, 1 << n)])
    keep = np.array([(mask >> k) & 1 for k in orders], dtype=bool)
    assert np.all(got[~keep] == 0.0)
    for c in range(0, B, 11):
        ref = oracle.o1_all_subsets(G[..., c], nf, sig, sb=sb)
        M = oracle.o1_all_subsets(G[..., c], nf, sig, sb=sb, absolute=True)
        assert np.all(np.abs(got[keep, c] - ref[keep]) <= 1e-10 * M[keep]), (c, got[keep, c], ref[keep])


@pytest.mark.gpu
@pytest.mark.parametrize("n,mask,with_q,B", [(2, 0, True, 5), (5, 0, True, 301), (8, (1 << 2) | (1 << 8), False, 4099),
                                             (8, 0, True, 64), (12, 1 << 12, True, 33)])
def test_flux_weights_vs_oracle(cos, n, mask, with_q, B):
    """cos_flux_weights against Eq. 6-7 written out (oracle.flux_weights); both sides add the subsets in increasing
    bitmask order with the same operations, so the comparison is to a few ulp of W."""
    import torch
    rng = np.random.default_rng(n * 100 + B)
    ns = (1 << n) - 1
    C = rng.standard_normal((ns, B)) * np.exp(rng.standard_normal((ns, 1)) * 3)
    Q = rng.random((ns, B)) if with_q else None
    lam = [0.0] + list(rng.standard_normal(n))
    Cd = torch.from_numpy(C).cuda()
    Qd = torch.from_numpy(Q).cuda() if with_q else None
    W = torch.empty(B, dtype=torch.float64, device="cuda")
    Phi = torch.full((ns, B), float("nan"), dtype=torch.float64, device="cuda")
    cos.cos_flux_weights(n, mask, lam, Cd, Qd, B, W, Phi)
    W2 = torch.empty(B, dtype=torch.float64, device="cuda")
    cos.cos_flux_weights(n, mask, lam, Cd, Qd, B, W2, None)
    torch.cuda.synchronize()
    Wh, Ph = W.cpu().numpy(), Phi.cpu().numpy()
    assert torch.equal(W, W2)
    for c in sorted(set([0, 1, B // 2, B - 1])):
        Wr, pr = oracle.flux_weights(C[:, c], None if Q is None else Q[:, c], lam, mask)
        assert np.array_equal(Ph[:, c], pr)
        assert abs(Wh[c] - Wr) <= 4e-16 * Wr * ns
    cos.cos_flux_weights(n, mask, lam, Cd, Qd, 0, W, None)          # empty batch is a no-op
    with pytest.raises(cos.CosError):
        cos.cos_flux_weights(13, 0, lam, Cd, Qd, B, W, None)


@pytest.mark.gpu
def test_envelope_to_weights_pipeline(cos):
    """tabulate -> all-subset readouts restricted to U = {2, 4} -> heat-bath weight, against O2a + Eq. 6-7 (cfg2-shaped,
    n = 6)."""
    import torch
    from cos_workloads import get_config, draw_vertices
    from cos_workloads.tables import table_for
    w = get_config(2).scaled(n=6, batch=70)
    table, v = table_for(w), draw_vertices(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    G = torch.empty((w.d * w.d, w.batch), dtype=torch.float64, device="cuda")
    cos.cos_tabulate(tab, w.n, torch.from_numpy(v["sites"]).cuda(), torch.from_numpy(v["tau"]).cuda(), w.batch, G)
    mask = (1 << 2) | (1 << 4)
    h = cos.cos_build_orders(w.n, 2, 0, None, mask)
    ns = (1 << w.n) - 1
    out = torch.empty((ns, w.batch), dtype=torch.float64, device="cuda")
    cos.cos_eval(h, G, w.batch, out)
    lam = [0.0, 1.0, -0.5, 0.25, 2.0, 1.0, 1.0]
    W = torch.empty(w.batch, dtype=torch.float64, device="cuda")
    cos.cos_flux_weights(w.n, mask, lam, out, None, w.batch, W, None)
    torch.cuda.synchronize()
    cos.cos_free(h); cos.cos_tab_free(tab)
    Gh = oracle.tabulate_reference(table, v["sites"], v["tau"])
    for c in (0, 37, 69):
        A = np.ascontiguousarray(Gh[0, :, :, c])
        Cref = oracle.o2a_twospin(A, A)
        Mref = oracle.o3_uniform(A, 2, 0.0, True, absolute=True)
        Wr, _ = oracle.flux_weights(Cref, None, lam, mask)
        Wm, _ = oracle.flux_weights(Mref, None, np.abs(lam), mask)
        assert abs(W[c].item() - Wr) <= 1e-10 * Wm
