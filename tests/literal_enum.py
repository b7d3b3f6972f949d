"""Independent, literal (pure Python) enumeration of connected typed contractions
Omega = (pi, Z, lambda), Eq. 58-63 — used ONLY to pin oracle/ on tiny n.

Deliberately different from oracle/cos_oracle.c: explicit colour assignments (no per-cycle
factorisation), sign by inversion count (not by cycle count), connectivity by graph search
(not union-find).
"""
import itertools


def _sign_by_inversions(p):
    inv = 0
    for i in range(len(p)):
        for j in range(i + 1, len(p)):
            if p[i] > p[j]:
                inv += 1
    return -1.0 if inv & 1 else 1.0


def _connected(p, n):
    N = 2 * n
    adj = {v: {p[v], (v + n) % N} for v in range(N)}
    for v in range(N):
        adj[p[v]].add(v)
    seen, stack = {0}, [0]
    while stack:
        v = stack.pop()
        for w in adj[v]:
            if w not in seen:
                seen.add(w)
                stack.append(w)
    return len(seen) == N


def _cycles(p):
    seen, out = set(), []
    for v in range(len(p)):
        if v in seen:
            continue
        c, w = [], v
        while w not in seen:
            seen.add(w)
            c.append(w)
            w = p[w]
        out.append(c)
    return out


def typed_connected_sum(A, sigma, n_flavors, absolute=False, distinct_colours_only=False):
    """S_n of Eq. 63.  A[lam][i][j] nested lists / arrays, sigma[lam] or None.
    absolute: sum |weight| instead.  distinct_colours_only: keep only the terms in which the two endpoints
    of every vertex that both lie in normal cycles have DIFFERENT colours (the terms Eq. 35 keeps)."""
    n = len(A[0])
    N = 2 * n
    total = 0.0
    for p in itertools.permutations(range(N)):
        if not _connected(p, n):
            continue
        sgn = _sign_by_inversions(p)
        cycles = _cycles(p)
        fixed = [c[0] for c in cycles if len(c) == 1]
        shift_sets = [()]
        if sigma is not None:
            shift_sets = itertools.chain.from_iterable(
                itertools.combinations(fixed, k) for k in range(len(fixed) + 1))
        for Z in shift_sets:
            Zs = set(Z)
            if any(((v + n) % N) in Zs for v in Zs):
                continue                          # matched shift pair: excluded (Eq. 83)
            normal = [c for c in cycles if not (len(c) == 1 and c[0] in Zs)]
            cyc_index = {}
            for ci, c in enumerate(normal):
                for v in c:
                    cyc_index[v] = ci
            for colours in itertools.product(range(n_flavors), repeat=len(normal)):
                if distinct_colours_only and any(
                        v in cyc_index and (v + n) in cyc_index and
                        colours[cyc_index[v]] == colours[cyc_index[v + n]] for v in range(n)):
                    continue
                w = sgn
                for ci, c in enumerate(normal):
                    lam = colours[ci]
                    for v in c:
                        w *= A[lam][v % n][p[v] % n]
                for v in Zs:
                    w *= sigma[colours[cyc_index[(v + n) % N]]]      # Eq. 60
                total += abs(w) if absolute else w
    return total


def uniform_connected_sum(A, n_flavors, sigma=0.0, absolute=False):
    """sum over connected pi of sgn(pi) N_f^{#cycles} prod A (Eq. 59).  With a counterterm (PAPER.md:431,
    reading G12) a true one-cycle v -> v is either a normal loop, N_f A[v][v], or a shift one-cycle, sigma (= N_f times the
    true-diagonal weight sigma/N_f); a vertex whose two endpoints are BOTH shift one-cycles is excluded (only possible
    at n = 1, Eq. 83).  absolute: every term enters with its absolute value -- the cancellation scale M of the
    uniform-mode tolerance (the normal and the shift choice of a one-cycle are separate terms)."""
    n = len(A)
    N = 2 * n
    total = 0.0
    for p in itertools.permutations(range(N)):
        if not _connected(p, n):
            continue
        sgn = _sign_by_inversions(p)
        cycles = _cycles(p)
        fixed = [c[0] for c in cycles if len(c) == 1]
        long_w = 1.0
        for c in cycles:
            if len(c) > 1:
                w = float(n_flavors)
                for v in c:
                    w *= A[v % n][p[v] % n]
                long_w *= w
        for k in range(len(fixed) + 1):
            for Z in itertools.combinations(fixed, k):
                if k and sigma == 0.0:
                    continue
                Zs = set(Z)
                if any(((v + n) % N) in Zs for v in Zs):
                    continue
                w = sgn * long_w
                for v in fixed:
                    w *= sigma if v in Zs else n_flavors * A[v % n][v % n]
                total += abs(w) if absolute else w
    return total
