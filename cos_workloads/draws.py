"""Seeded vertex configurations and random test matrices (inputs only)."""
import numpy as np


def draw_vertices(w, batch=None):
    """Recipe of SURVEY.md 8(d): NumPy default_rng(seed); in this order
    sites = integers(0, L, (B, n, 2)); [honeycomb: sub = integers(0, 2, (B, n))];
    tau = random((B, n)) * beta.

    Returns a dict of batch-innermost arrays (the device layout):
        sites int32 [n][2][B], tau fp64 [n][B], sub int32 [n][B] (honeycomb only; the
        sublattice-summed DAG ignores it — reading G20).
    """
    B = w.batch if batch is None else int(batch)
    rng = np.random.default_rng(w.seed)
    sites = rng.integers(0, w.L, size=(B, w.n, 2))
    out = {}
    if w.lattice == 1:
        sub = rng.integers(0, 2, size=(B, w.n))
        out["sub"] = np.ascontiguousarray(sub.transpose(1, 0).astype(np.int32))
    tau = rng.random((B, w.n)) * w.beta
    out["sites"] = np.ascontiguousarray(sites.transpose(1, 2, 0).astype(np.int32))
    out["tau"] = np.ascontiguousarray(tau.transpose(1, 0).astype(np.float64))
    return out


def draw_clustered_vertices(w, batch=None, spread=1, tau_window=None):
    """Stress input: the vertices of a configuration sit within +-`spread` sites of a random
    centre and within a tau window of `tau_window` (default beta/50) around a random time -- the short-distance,
    short-time clusters a sampler of the paper's kind visits, where the terms of the connected sum
    cancel hardest.  Same layout as draw_vertices; seeded with w.seed + 7919."""
    B = w.batch if batch is None else int(batch)
    win = w.beta / 50.0 if tau_window is None else float(tau_window)
    rng = np.random.default_rng(w.seed + 7919)
    centre = rng.integers(0, w.L, size=(B, 1, 2))
    sites = (centre + rng.integers(-spread, spread + 1, size=(B, w.n, 2))) % w.L
    t0 = rng.random((B, 1)) * (w.beta - win)
    tau = t0 + rng.random((B, w.n)) * win
    out = {}
    if w.lattice == 1:
        out["sub"] = np.ascontiguousarray(rng.integers(0, 2, size=(B, w.n)).transpose(1, 0).astype(np.int32))
    out["sites"] = np.ascontiguousarray(sites.transpose(1, 2, 0).astype(np.int32))
    out["tau"] = np.ascontiguousarray(tau.transpose(1, 0).astype(np.float64))
    return out


def random_matrices(seed, n_blocks, d, batch, scale=1.0, diag=None):
    """Generic propagator blocks G[n_blocks][d][d][batch] ~ scale * N(0, 1) (unit tests).
    `diag` (float) overrides the diagonal, mimicking g(0, 0^-) = -rho."""
    rng = np.random.default_rng(seed)
    G = rng.standard_normal((n_blocks, d, d, batch)) * scale
    if diag is not None:
        for a in range(d):
            G[:, a, a, :] = diag * (1.0 + 0.1 * rng.standard_normal((n_blocks, batch)))
    return np.ascontiguousarray(G)
