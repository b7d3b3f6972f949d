"""Pins for the synthetic inputs (cos_workloads) and the oracle of the tabulation step A2 (CPU only)."""
import numpy as np
import pytest

import oracle
from cos_workloads import CONFIGS, build_table, draw_vertices, get_config
from cos_workloads.tables import table_for


def _direct_square(L, t, mu, beta, r, tau):
    """g(r, tau) by the explicit k-sum, 0 < tau < beta (independent of the FFT used by build_table)."""
    acc = 0.0
    for kx in range(L):
        for ky in range(L):
            xi = -2 * t * (np.cos(2 * np.pi * kx / L) + np.cos(2 * np.pi * ky / L)) - mu
            ph = np.cos(2 * np.pi * (kx * r[0] + ky * r[1]) / L)
            acc += ph * np.exp(-xi * tau) / (1 + np.exp(-beta * xi))
    return acc / (L * L)


def test_square_table_matches_direct_ksum_and_sum_rule():
    L, t, mu, beta, nt = 6, 1.0, -0.3, 2.0, 65
    T = build_table(0, L, t, (mu,), beta, nt)
    for r in ((0, 0), (1, 0), (2, 5)):
        for k in (0, 7, nt - 1):
            tau = k * beta / (nt - 1)
            assert abs(T.data[0, 0, r[0] * L + r[1], k] - _direct_square(L, t, mu, beta, r, tau)) < 1e-13
    # g(r, 0+) + g(r, beta-) = delta_{r,0}   (anticommutator)
    s = T.data[0, 0, :, 0] + T.data[0, 0, :, -1]
    assert abs(s[0] - 1.0) < 1e-13 and np.max(np.abs(s[1:])) < 1e-13


def test_half_filling_density():
    """mu = 0 on the bipartite square lattice: rho = 1/2, so g(0, 0^-) = -1/2."""
    T = build_table(0, 8, 1.0, (0.0,), 2.0, 33)
    assert abs(T.data[0, 0, 0, -1] - 0.5) < 1e-13


def test_honeycomb_table_sum_rule_and_symmetry():
    L, beta, nt = 6, 3.0, 17
    T = build_table(1, L, 1.0, (0.3, -0.3), beta, nt)
    assert T.data.shape == (2, 4, L * L, nt)
    for b in range(2):
        for ss in range(4):
            s = T.data[b, ss, :, 0] + T.data[b, ss, :, -1]
            expect0 = 1.0 if ss in (0, 3) else 0.0
            assert abs(s[0] - expect0) < 1e-13 and np.max(np.abs(s[1:])) < 1e-13
        # g^{AB}(R) = g^{BA}(-R)
        for dx in range(L):
            for dy in range(L):
                a = T.data[b, 1, dx * L + dy]
                c = T.data[b, 2, ((-dx) % L) * L + ((-dy) % L)]
                assert np.max(np.abs(a - c)) < 1e-13
    # mu = 0 honeycomb is half filled; mu_eff = +-0.3 moves the density symmetrically
    rho = T.data[:, 0, 0, -1]
    assert abs(rho[0] + rho[1] - 1.0) < 1e-12 and rho[0] > 0.5 > rho[1]


def test_draws_are_seeded_and_batch_innermost():
    w = get_config(3).scaled(batch=16)
    a, b = draw_vertices(w), draw_vertices(w)
    assert a["sites"].shape == (w.n, 2, 16) and a["tau"].shape == (w.n, 16) and a["sub"].shape == (w.n, 16)
    assert np.array_equal(a["sites"], b["sites"]) and np.array_equal(a["tau"], b["tau"])
    assert a["sites"].min() >= 0 and a["sites"].max() < w.L
    assert a["tau"].min() >= 0 and a["tau"].max() < w.beta
    assert [c.n for c in CONFIGS] == [4, 8, 10, 10, 12]
    assert [c.batch for c in CONFIGS] == [1024, 65536, 16384, 8192, 64]


def test_tabulation_reference_conventions():
    """Readings G17-G18: anti-periodic sign, 0^- on the diagonal, exact at nodes, O(dtau^2) lerp error."""
    w = get_config(1)
    T = table_for(w)
    v = draw_vertices(w, batch=32)
    G = oracle.tabulate_reference(T, v["sites"], v["tau"])
    assert G.shape == (1, w.n, w.n, 32)
    rho = T.data[0, 0, 0, -1]
    assert np.allclose(G[0, np.arange(w.n), np.arange(w.n), :], -rho, rtol=0, atol=1e-15)
    # entry (i, j) against the direct k-sum
    for (i, j, b) in ((0, 1, 0), (2, 3, 5), (3, 0, 7)):
        dt = v["tau"][i, b] - v["tau"][j, b]
        sign = 1.0
        if dt <= 0:
            dt += w.beta
            sign = -1.0
        r = ((v["sites"][i, 0, b] - v["sites"][j, 0, b]) % w.L, (v["sites"][i, 1, b] - v["sites"][j, 1, b]) % w.L)
        exact = sign * _direct_square(w.L, w.t, w.mu, w.beta, r, dt)
        assert abs(G[0, i, j, b] - exact) < 5e-5          # (beta/1023)^2/8 * max|g''| ~ 1e-5
    # exactly on a node the interpolation returns the node value
    tau = np.zeros((w.n, 1))
    step = w.beta / (w.n_tau - 1)
    tau[1, 0] = 100 * step
    sites = np.zeros((w.n, 2, 1), dtype=np.int32)
    G1 = oracle.tabulate_reference(T, sites, tau)
    assert abs(G1[0, 1, 0, 0] - T.data[0, 0, 0, 100]) < 1e-14
    assert abs(G1[0, 0, 1, 0] + T.data[0, 0, 0, w.n_tau - 1 - 100]) < 1e-12      # -g(beta - 100 step)
    # equal times between distinct vertices also use 0^-  (dt = 0 -> beta, sign -)
    assert abs(G1[0, 2, 3, 0] + T.data[0, 0, 0, -1]) < 1e-15


def test_tabulation_reference_honeycomb_layout():
    w = get_config(3).scaled(n=3, batch=4)
    T = table_for(w)
    v = draw_vertices(w)
    G = oracle.tabulate_reference(T, v["sites"], v["tau"])
    assert G.shape == (2, 6, 6, 4)
    # endpoint index a = i * n_sub + s; same vertex, different sublattice, equal time -> -g^{AB}(0, beta)
    assert np.allclose(G[1, 0, 1, :], -T.data[1, 1, 0, -1])
    assert np.allclose(G[1, 1, 0, :], -T.data[1, 2, 0, -1])
