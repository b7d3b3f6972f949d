"""ctypes front-end of the CPU oracle (oracle/cos_oracle.c) plus the NumPy reference of the
propagator tabulation step.  TEST INFRASTRUCTURE ONLY (see the C file's header).

All functions take ONE configuration; `G` is that configuration's propagator blocks
G[n_blocks][d][d] with d = n * n_sub and endpoint index a = i * n_sub + s
(from-endpoint first, Eq. 59 / reading G7).
"""
import ctypes
import itertools
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cos_oracle.c")
_LIB = os.path.join(_HERE, "libcos_oracle.so")
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_llp = ctypes.POINTER(ctypes.c_longlong)


def build_oracle(force=False):
    """gcc -O2 the oracle into oracle/libcos_oracle.so (idempotent)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=gnu99", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build_oracle())
        lib.cos_o1_connected.restype = ctypes.c_double
        lib.cos_o1_connected.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp, _dp, ctypes.c_int]
        lib.cos_o2a_twospin.restype = ctypes.c_int
        lib.cos_o2a_twospin.argtypes = [ctypes.c_int, _dp, _dp, ctypes.c_double, ctypes.c_double, ctypes.c_int, _dp]
        lib.cos_o2b_polynomial.restype = ctypes.c_int
        lib.cos_o2b_polynomial.argtypes = [ctypes.c_int, ctypes.c_int, _dp, _dp, ctypes.c_int, _dp]
        lib.cos_o3_alg3.restype = ctypes.c_double
        lib.cos_o3_alg3.argtypes = [ctypes.c_int, ctypes.c_int, _dp, _dp, ctypes.c_int, _llp, _llp]
        lib.cos_o3_uniform.restype = ctypes.c_int
        lib.cos_o3_uniform.argtypes = [ctypes.c_int, ctypes.c_int, _dp, ctypes.c_double, ctypes.c_int,
                                       ctypes.c_int, _dp, _llp, _llp]
        _lib = lib
    return _lib


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _sig(sigma):
    if sigma is None:
        return None, None
    s = np.ascontiguousarray(np.atleast_1d(sigma), dtype=np.float64)
    return s, s.ctypes.data_as(_dp)


# ------------------------------------------------------------------ single-block-set routines
def o1_connected(A, n_flavors, sigma=None, sb=True, absolute=False):
    """Brute-force definition Eq. 58-63 on A[nb][n][n] (nb = N_f if sb else 1)."""
    A, pA = _c(A)
    n = A.shape[-1]
    assert A.shape == ((n_flavors if sb else 1), n, n)
    s, ps = _sig(sigma)
    return _load().cos_o1_connected(n, n_flavors, int(sb), pA, ps, int(absolute))


def o2a_twospin(A_up, A_dn, sig_up=0.0, sig_dn=0.0, absolute=False):
    """Two-spin determinants + CDet (Eq. 49-50, 53): all 2^n - 1 connected values (binary128 inside).
    absolute=True: permanents of |A|, |sigma| -- a LOWER bound of the cancellation scale M (C file, O2 header)."""
    A_up, pu = _c(A_up)
    A_dn, pd = _c(A_dn)
    n = A_up.shape[0]
    out = np.zeros((1 << n) - 1)
    rc = _load().cos_o2a_twospin(n, pu, pd, float(sig_up), float(sig_dn), int(absolute), out.ctypes.data_as(_dp))
    assert rc == 0
    return out


def o2b_polynomial(A, sigma=None, absolute=False):
    """Flavour-polynomial route Eq. 34-38 on A[N_f][n][n]: all 2^n - 1 connected values (binary128 inside).
    absolute=True: permanents of |A|, |sigma| -- a LOWER bound of the cancellation scale M (C file, O2 header).
    absolute=2: additionally every minus sign of Eq. 38 becomes a plus -- the rounding-error scale of evaluating the
    ROUTE in floating point (it keeps the disconnected products Eq. 38 subtracts); tolerance scale of cos_det_eval."""
    A, pA = _c(A)
    nf, n, _ = A.shape
    s, ps = _sig(sigma)
    out = np.zeros((1 << n) - 1)
    rc = _load().cos_o2b_polynomial(n, nf, pA, ps, int(absolute), out.ctypes.data_as(_dp))
    assert rc == 0
    return out


def o3_alg3(A, sigma=None, absolute=False, counts=False):
    """Literal Algorithm 3 on A[N_f][n][n]."""
    A, pA = _c(A)
    nf, n, _ = A.shape
    s, ps = _sig(sigma)
    ns, nu = ctypes.c_longlong(0), ctypes.c_longlong(0)
    v = _load().cos_o3_alg3(n, nf, pA, ps, int(absolute), ctypes.byref(ns), ctypes.byref(nu))
    return (v, ns.value, nu.value) if counts else v


def o3_uniform(A, n_flavors, sigma=0.0, all_subsets=False, absolute=False, counts=False):
    """Uniform rooted recurrence Eq. 8-15 on A[n][n]; returns [1] or [2^n - 1] values."""
    A, pA = _c(A)
    n = A.shape[-1]
    out = np.zeros((1 << n) - 1 if all_subsets else 1)
    ns, nu = ctypes.c_longlong(0), ctypes.c_longlong(0)
    rc = _load().cos_o3_uniform(n, n_flavors, pA, float(sigma), int(all_subsets), int(absolute),
                                out.ctypes.data_as(_dp), ctypes.byref(ns), ctypes.byref(nu))
    assert rc == 0
    return (out, ns.value, nu.value) if counts else out


# ------------------------------------------------------------------ subsets and sublattice sums
def subset_blocks(G, verts, assign, n_sub):
    """A[lam][a][b] = G[lam][(verts[a], assign[a])][(verts[b], assign[b])]  (principal sub-block of
    the envelope matrix, at fixed sublattice assignment, Eq. 54-55)."""
    idx = [v * n_sub + s for v, s in zip(verts, assign)]
    return np.ascontiguousarray(G[:, idx][:, :, idx])


def o1_all_subsets(G, n_flavors, sigma=None, sb=True, absolute=False):
    """Definition-level all-subset values on a square-lattice block set G[nb][n][n]."""
    n = G.shape[-1]
    out = np.zeros((1 << n) - 1)
    for S in range(1, 1 << n):
        verts = [i for i in range(n) if S >> i & 1]
        out[S - 1] = o1_connected(subset_blocks(G, verts, [0] * len(verts), 1), n_flavors, sigma, sb, absolute)
    return out


def connected_reference(G, n, n_sub, n_flavors, sigmas=None, uniform=True, all_subsets=False,
                        tier="o1", absolute=False):
    """Reference output vector of ONE configuration, in the C-ABI's output order
    (index 0 = full set if not all_subsets, else index bitmask(S) - 1).

    Sublattice-summed (Eq. 55): C_S = sum over assignments s in [n_sub]^{|S|} of the connected
    sum of A^{(s)}[S, S].   tier: 'o1' brute force, 'o3' printed recurrences,
    'o2a' two-spin determinants (N_f = 2), 'o2b' polynomial route (SB, any N_f).
    """
    G = np.asarray(G, dtype=np.float64)
    subsets = range(1, 1 << n) if all_subsets else [(1 << n) - 1]
    out = np.zeros(len(subsets))
    for k, S in enumerate(subsets):
        verts = [i for i in range(n) if S >> i & 1]
        acc = 0.0
        for assign in itertools.product(range(n_sub), repeat=len(verts)):
            A = subset_blocks(G, verts, assign, n_sub)
            if tier == "o1":
                sig = sigmas if not uniform else (None if sigmas is None else [float(np.atleast_1d(sigmas)[0])])
                acc += o1_connected(A, n_flavors, sig, sb=not uniform, absolute=absolute)
            elif tier == "o3":
                if uniform:
                    s0 = 0.0 if sigmas is None else float(np.atleast_1d(sigmas)[0])
                    acc += o3_uniform(A[0], n_flavors, s0, False, absolute)[0]
                else:
                    acc += o3_alg3(A, sigmas, absolute)
            elif tier == "o2a":
                assert n_flavors == 2
                if uniform:
                    assert sigmas is None
                    acc += o2a_twospin(A[0], A[0], absolute=absolute)[-1]
                else:
                    sg = (0.0, 0.0) if sigmas is None else sigmas
                    acc += o2a_twospin(A[0], A[1], sg[0], sg[1], absolute=absolute)[-1]
            elif tier == "o2b":
                assert not uniform
                acc += o2b_polynomial(A, sigmas, absolute=absolute)[-1]
            else:
                raise ValueError(tier)
        out[k] = acc
    return out


# ------------------------------------------------------------------ tabulation step (A2) reference
def tabulate_reference(table, sites, tau):
    """Propagator tabulation by linear interpolation (readings G17-G18):
        A[(i,s),(j,s')] = sign * lerp(T^{ss'}[r_i - r_j mod L], dtau),  dtau = tau_i - tau_j,
        dtau <= 0  ->  dtau += beta, sign = -1   (anti-periodicity; equal time and i = j use 0^-,
        so the diagonal is g(0, 0^-) = -rho);
        nodes tau_k = k beta/(n_tau-1): u = dtau/step, k = min(floor(u), n_tau-2), w = u-k,
        g = (1-w) T_k + w T_{k+1}.
    table: cos_workloads.PropTable; sites int [n][2][B]; tau fp64 [n][B].
    Returns G[n_blocks][d][d][B] (batch innermost)."""
    T = table.data
    nb, L, ns, nt, beta = T.shape[0], table.L, table.n_sub, table.n_tau, table.beta
    n, _, B = sites.shape
    d = n * ns
    step = beta / (nt - 1)
    G = np.zeros((nb, d, d, B))
    cols = np.arange(B)
    for i in range(n):
        for j in range(n):
            dx = (sites[i, 0] - sites[j, 0]) % L
            dy = (sites[i, 1] - sites[j, 1]) % L
            r = dx * L + dy
            dt = tau[i] - tau[j]
            neg = dt <= 0.0
            dt = np.where(neg, dt + beta, dt)
            sign = np.where(neg, -1.0, 1.0)
            u = dt / step
            k = np.minimum(np.floor(u).astype(np.int64), nt - 2)
            w = u - k
            for lam in range(nb):
                for s in range(ns):
                    for s2 in range(ns):
                        tab = T[lam, s * ns + s2]
                        g = (1.0 - w) * tab[r, k] + w * tab[r, k + 1]
                        G[lam, i * ns + s, j * ns + s2, cols] = sign * g
    return G


# ------------------------------------------------------------------ many-configuration weights (Eq. 6-7)
def flux_weights(C, Q, lambdas, order_mask=0):
    """Signed fluxes and heat-bath normalisation of ONE envelope, written out from PAPER.md:106-113:
        Phi_S = lambda_{|S|} C_{|S|}(V_S) Q_{S-bar|S}          for |S| in the allowed orders U     (Eq. 6)
        W     = sum_{S subset [N], |S| in U} |Phi_S| / binom(N, |S|)                              (Eq. 7)
    C, Q: arrays [2^N - 1] indexed by bitmask(S) - 1 (Q None -> 1); lambdas[k] = lambda_k, k = 0..N;
    order_mask bit k <-> k in U (0 = every order).  Returns (W, Phi[2^N - 1]) with Phi = 0 outside U."""
    import math
    C = np.asarray(C, dtype=np.float64)
    N = int(round(math.log2(C.shape[0] + 1)))
    assert (1 << N) - 1 == C.shape[0]
    phi = np.zeros_like(C)
    W = 0.0
    for S in range(1, 1 << N):
        k = bin(S).count("1")
        if order_mask and not (order_mask >> k) & 1:
            continue
        p = lambdas[k] * C[S - 1]
        if Q is not None:
            p = p * Q[S - 1]
        phi[S - 1] = p
        W += abs(p) / math.comb(N, k)
    return W, phi
