/*
 * cos_oracle.c -- CPU ORACLE for the CoS / SB-CoS connected sums of arxiv 2507.12349.
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct C written from the paper
 * (/root/reference/PAPER.md, cited as PAPER.md:<line>).  It shares NO code, header,
 * table or helper with the CUDA path under paper_2507_12349_b200/ and is never called
 * by the product path.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.
 *
 * Tiers:
 *   O1  the DEFINITION: sum over all permutations of the 2n endpoints, connected ones kept
 *       by union-find over fermion edges plus interaction lines, explicit shift one-cycles,
 *       colour sums (Eq. 58-63; uniform: PAPER.md:45, 431).
 *   O2a two-spin determinant route + CDet subset recursion (Eq. 49-50,
 *       446-450 Eq. 53), __float128 (the paper needs double-double there).
 *   O2b flavour-polynomial route, Eq. 34-38, __float128.
 *   O3  the recurrences as printed: Algorithm 3 (canonical key Eq. 79-80)
 *       and the uniform rooted recurrence with all-subset readouts (Eq. 8-15).
 *
 * Matrix convention everywhere: A[lam][i][j], row-major n x n per flavour block,
 * A[i][j] = propagator from endpoint residue i to endpoint residue j (Eq. 59: A[vbar, pi(v)bar]).
 * Vertices / flavours are 0-based here (1-based in the paper).
 *
 * `absolute` != 0 evaluates the same sum with |A|, |sigma| and every sign dropped: the
 * cancellation bound M of the acceptance test |GPU - oracle| <= 1e-10 * M (BASELINE.json).
 *
 * Pins: see tests/test_oracle_pins.py (closed forms Eq. 83, hand-computed n<=2 values,
 * O1 == O2a == O2b == O3 on random inputs, literal colour enumeration in Python).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define MAXN 12
#define MAXV (2 * MAXN)
#define MAXF 8

static double absd(double x, int absolute) { return absolute ? fabs(x) : x; }

/* ------------------------------------------------------------------------------------------
 * O1: brute-force definition.
 * ---------------------------------------------------------------------------------------- */

typedef struct {
    int n, N, nf, sb, absolute, has_shift;
    const double *A;      /* [nb][n][n], nb = sb ? nf : 1 */
    const double *sigma;  /* [nb] or NULL */
    int perm[MAXV];
    int used[MAXV];
    double total;
} o1_ctx;

static int uf_find(int *p, int x) { while (p[x] != x) { p[x] = p[p[x]]; x = p[x]; } return x; }

/* Weight of one permutation: sgn(pi) * sum over admissible shift sets Z and colourings
 * (Eq. 62), colour sum factorised per normal cycle:  prod_C [ sum_lam sigma_lam^{k_C} prod_{v in C} A_lam ].
 * Uniform mode: each normal cycle carries N_f; a shift one-cycle carries sigma
 * (true-diagonal weight sigma/N_f times the closing N_f).                        */
static double o1_perm_weight(o1_ctx *c)
{
    const int n = c->n, N = c->N, nb = c->sb ? c->nf : 1;
    int i, v;
    /* connectivity of G(pi): edges {v, pi(v)} and {v, P(v)} (Eq. 61) */
    int uf[MAXV];
    for (v = 0; v < N; ++v) uf[v] = v;
    for (v = 0; v < N; ++v) {
        int a = uf_find(uf, v), b = uf_find(uf, c->perm[v]);
        if (a != b) uf[a] = b;
    }
    for (v = 0; v < n; ++v) {
        int a = uf_find(uf, v), b = uf_find(uf, v + n);
        if (a != b) uf[a] = b;
    }
    {
        int root = uf_find(uf, 0);
        for (v = 1; v < N; ++v) if (uf_find(uf, v) != root) return 0.0;
    }
    /* cycle decomposition */
    int cyc_of[MAXV], ncyc = 0, cyc_len[MAXV];
    double cyc_prod[MAXV][MAXF];
    for (v = 0; v < N; ++v) cyc_of[v] = -1;
    for (v = 0; v < N; ++v) {
        if (cyc_of[v] >= 0) continue;
        int w = v, len = 0, l;
        for (l = 0; l < nb; ++l) cyc_prod[ncyc][l] = 1.0;
        do {
            cyc_of[w] = ncyc;
            int nx = c->perm[w];
            for (l = 0; l < nb; ++l)
                cyc_prod[ncyc][l] *= absd(c->A[(l * n + (w % n)) * n + (nx % n)], c->absolute);
            w = nx; ++len;
        } while (w != v);
        cyc_len[ncyc] = len;
        ++ncyc;
    }
    double sgn = ((N - ncyc) & 1) ? -1.0 : 1.0;      /* sgn(pi) = (-1)^{2n-k} (Eq. 78) */
    if (c->absolute) sgn = 1.0;
    /* fixed points that may become shift cycles */
    int fix[MAXV], nfix = 0;
    if (c->has_shift)
        for (v = 0; v < N; ++v) if (c->perm[v] == v) fix[nfix++] = v;
    double sum = 0.0;
    uint32_t Z;
    for (Z = 0; Z < (1u << nfix); ++Z) {
        int is_shift[MAXV], kC[MAXV], ok = 1;
        memset(is_shift, 0, sizeof is_shift);
        memset(kC, 0, sizeof kC);
        for (i = 0; i < nfix; ++i) if (Z >> i & 1) is_shift[fix[i]] = 1;
        /* a shift {v} needs P(v) in a NORMAL cycle (Eq. 60); matched shift pairs are excluded
         * (PAPER.md:621 for n >= 2; physical convention Eq. 83 at n = 1)                       */
        for (v = 0; v < N && ok; ++v) if (is_shift[v]) {
            int p = (v + n) % N;
            if (is_shift[p]) ok = 0; else kC[cyc_of[p]] += 1;
        }
        if (!ok) continue;
        double w = sgn;
        int cy;
        for (cy = 0; cy < ncyc; ++cy) {
            /* is this cycle a shift one-cycle? */
            int shifted = 0;
            if (cyc_len[cy] == 1) for (v = 0; v < N; ++v) if (cyc_of[v] == cy && is_shift[v]) shifted = 1;
            if (shifted) continue;                    /* its sigma factor is charged to the partner's cycle */
            if (c->sb) {
                double s = 0.0; int l, k;
                for (l = 0; l < nb; ++l) {
                    double t = cyc_prod[cy][l];
                    for (k = 0; k < kC[cy]; ++k) t *= absd(c->sigma[l], c->absolute);
                    s += t;
                }
                w *= s;
            } else {
                double t = (double)c->nf * cyc_prod[cy][0]; int k;
                for (k = 0; k < kC[cy]; ++k) t *= absd(c->sigma[0], c->absolute);
                w *= t;
            }
        }
        sum += w;
    }
    return sum;
}

static void o1_rec(o1_ctx *c, int pos)
{
    if (pos == c->N) { c->total += o1_perm_weight(c); return; }
    int w;
    for (w = 0; w < c->N; ++w) {
        if (c->used[w]) continue;
        c->used[w] = 1; c->perm[pos] = w;
        o1_rec(c, pos + 1);
        c->used[w] = 0;
    }
}

/* S_n of Eq. 63 (sb != 0: SB-CoS, A has nf blocks, sigma may be NULL = no shifts) or the
 * uniform loop-factor sum (sb == 0: one block, factor nf per loop, sigma NULL or 1 value).    */
double cos_o1_connected(int n, int nf, int sb, const double *A, const double *sigma, int absolute)
{
    if (n < 1 || n > MAXN || nf < 1 || nf > MAXF) return NAN;
    o1_ctx c;
    memset(&c, 0, sizeof c);
    c.n = n; c.N = 2 * n; c.nf = nf; c.sb = sb; c.absolute = absolute;
    c.A = A; c.sigma = sigma; c.has_shift = (sigma != NULL);
    c.total = 0.0;
    o1_rec(&c, 0);
    return c.total;
}

/* ------------------------------------------------------------------------------------------
 * O2: determinant routes.  Arithmetic type: __float128 (IEEE binary128, eps = 2^-113, gcc soft
 * float).  The paper itself needs double-double for the determinant recursion: the
 * subset recursion Eq. 53 / Eq. 38 subtracts products of disconnected parts whose magnitude
 * c~(V) ~ (|V|-1)! prod_i a({i}) exceeds the connected value by > 10 orders at n = 10 on the
 * benchmark inputs (|C| ~ 1e-15, c~ ~ 1e6), so x87 long double (eps = 5e-20) is NOT enough there.
 *
 * `absolute` != 0 replaces every determinant by the PERMANENT of the element-wise absolute matrix
 * and sigma by |sigma| (same recursion): the sum of |weight| over the connected contractions this
 * route enumerates, i.e. those in which the two endpoints of a vertex lie in cycles of DIFFERENT
 * colour (Eq. 35 has no same-colour entry: those terms cancel identically in the signed sum,
 * PAPER.md:291-296).  It is therefore a LOWER bound of the full cancellation scale M of O1 / O3
 * with absolute = 1 (which also counts same-colour terms), used as a stricter acceptance scale
 * where O1 / O3 are too slow.
 * ---------------------------------------------------------------------------------------- */
typedef __float128 xreal;
static xreal xabs(xreal x) { return x < 0 ? -x : x; }

/* det of the principal submatrix A[T,T] + diag_add * 1, Gaussian elimination, partial pivoting */
static xreal x_minor(int n, const double *A, uint32_t T, double diag_add)
{
    xreal M[MAXN][MAXN];
    int idx[MAXN], k = 0, i, j, p;
    for (i = 0; i < n; ++i) if (T >> i & 1) idx[k++] = i;
    if (k == 0) return 1;
    for (i = 0; i < k; ++i)
        for (j = 0; j < k; ++j)
            M[i][j] = (xreal)A[idx[i] * n + idx[j]] + (i == j ? (xreal)diag_add : (xreal)0);
    xreal det = 1;
    for (p = 0; p < k; ++p) {
        int piv = p;
        for (i = p + 1; i < k; ++i) if (xabs(M[i][p]) > xabs(M[piv][p])) piv = i;
        if (M[piv][p] == 0) return 0;
        if (piv != p) {
            for (j = 0; j < k; ++j) { xreal t = M[p][j]; M[p][j] = M[piv][j]; M[piv][j] = t; }
            det = -det;
        }
        det *= M[p][p];
        for (i = p + 1; i < k; ++i) {
            xreal f = M[i][p] / M[p][p];
            for (j = p; j < k; ++j) M[i][j] -= f * M[p][j];
        }
    }
    return det;
}

/* permanent of |A[T,T]| + |diag_add| * 1 by its definition, expanded row by row over the set of
 * columns already used:  P_r[cols] = sum_{j in cols} |M[r][j]| * P_{r-1}[cols \ j]  (k 2^k terms). */
static xreal x_perm_abs(int n, const double *A, uint32_t T, double diag_add)
{
    int idx[MAXN], k = 0, i, j;
    for (i = 0; i < n; ++i) if (T >> i & 1) idx[k++] = i;
    if (k == 0) return 1;
    static __thread xreal P[1u << MAXN];          /* binary128: the subset recursion cancels as hard as for det */
    uint32_t cols, fullc = 1u << k;
    P[0] = 1;
    for (cols = 1; cols < fullc; ++cols) {
        int r = __builtin_popcount(cols) - 1;         /* rows 0..r are matched with the columns in cols */
        xreal acc = 0;
        for (j = 0; j < k; ++j)
            if (cols >> j & 1) {
                xreal m = (xreal)fabs(A[idx[r] * n + idx[j]]) + (r == j ? (xreal)fabs(diag_add) : (xreal)0);
                acc += m * P[cols ^ (1u << j)];
            }
        P[cols] = acc;
    }
    return P[fullc - 1];
}

static xreal x_minor_or_perm(int n, const double *A, uint32_t T, double diag_add, int absolute)
{
    return absolute ? x_perm_abs(n, A, T, diag_add) : x_minor(n, A, T, diag_add);
}

static int popc(uint32_t x) { return __builtin_popcount(x); }

/* CDet recursion Eq. 53 / Eq. 38: c(V) = a(V) - sum over PROPER subsets
 * S of V containing min V of c(S) a(V \ S); a(empty) = 1; increasing subset size.
 * a, c are arrays over bitmasks [2^n]; c[0] unused.                                              */
static void cdet_recursion(int n, const xreal *a, xreal *c)
{
    uint32_t full = (1u << n), V;
    int size;
    c[0] = 0;
    for (size = 1; size <= n; ++size)
        for (V = 1; V < full; ++V) {
            if (popc(V) != size) continue;
            uint32_t anchor = V & (~V + 1u);          /* lowest set bit = min V */
            uint32_t rest = V ^ anchor, sub;
            xreal acc = a[V];
            /* S = anchor | sub, sub a PROPER subset of rest (so that S != V) */
            for (sub = (rest - 1) & rest; ; sub = (sub - 1) & rest) {
                if (rest == 0) break;
                uint32_t S = anchor | sub;
                acc -= c[S] * a[V ^ S];
                if (sub == 0) break;
            }
            c[V] = acc;
        }
}

/* Rounding-error scale of a floating-point evaluation of Eq. 53 / Eq. 38 itself (not of the connected value): the same
 * recursion with every term taken positive, R(V) = a(V) + sum_S R(S) a(V \ S), on a >= 0 (the moments evaluated on
 * |A|, |sigma|).  It contains the disconnected products that the recursion subtracts, so R >= |c|; it bounds what an
 * fp64 evaluation of the determinant route can lose, and is used only as the tolerance scale of that route's tests
 * (cos_o2b_polynomial with absolute = 2).                                                            */
static void cdet_route_scale(int n, const xreal *a, xreal *c)
{
    uint32_t full = (1u << n), V;
    int size;
    c[0] = 0;
    for (size = 1; size <= n; ++size)
        for (V = 1; V < full; ++V) {
            if (popc(V) != size) continue;
            uint32_t anchor = V & (~V + 1u);
            uint32_t rest = V ^ anchor, sub;
            xreal acc = a[V];
            for (sub = (rest - 1) & rest; ; sub = (sub - 1) & rest) {
                if (rest == 0) break;
                acc += c[anchor | sub] * a[V ^ (anchor | sub)];
                if (sub == 0) break;
            }
            c[V] = acc;
        }
}

/* O2a / O2a': two-spin Hubbard.  Full contraction sum at fixed vertices = product of two
 * determinants; the counterterm enters the TRUE diagonal of spin s with the
 * OPPOSITE spin's weight (Eq. 49); 2 endpoint assignments per contact vertex:
 *   a(T) = 2^{|T|} det(A_up[T] + sig_dn 1) det(A_dn[T] + sig_up 1),   c by Eq. 53,
 * and the scalar term of Eq. 50 is removed from singletons: C({i}) = c({i}) - 2 sig_up sig_dn.
 * out[T-1] = C(T) for every nonempty T (bit i <-> vertex i).                                     */
int cos_o2a_twospin(int n, const double *A_up, const double *A_dn, double sig_up, double sig_dn, int absolute,
                    double *out)
{
    if (n < 1 || n > MAXN) return 1;
    uint32_t full = 1u << n, T;
    xreal *a = (xreal *)malloc(sizeof(xreal) * full);
    xreal *c = (xreal *)malloc(sizeof(xreal) * full);
    if (!a || !c) { free(a); free(c); return 2; }
    a[0] = 1;
    for (T = 1; T < full; ++T)
        a[T] = (xreal)(double)(1u << popc(T)) * x_minor_or_perm(n, A_up, T, sig_dn, absolute) *
               x_minor_or_perm(n, A_dn, T, sig_up, absolute);
    cdet_recursion(n, a, c);
    for (T = 1; T < full; ++T) {
        xreal v = c[T];
        if (popc(T) == 1) v -= (xreal)2 * (xreal)absd(sig_up, absolute) * (xreal)absd(sig_dn, absolute);
        out[T - 1] = (double)v;
    }
    free(a); free(c);
    return 0;
}

/* O2b: flavour-polynomial route, Eq. 34-38, for any N_f (reading G13 of SURVEY.md generalises
 * the three-flavour tensor Eq. 35: a site carried by no flavour is not in T; by exactly one
 * flavour a -> 2 sigma_a; by exactly two flavours a<b -> 2; by three or more -> 0).
 *   d_a(S) = det A_a[S,S]                                  (Eq. 34)
 *   H(T)   = sum over local choices of prod_a d_a(S_a) prod_i L_i   (Eq. 36)
 *   C(T)   = H(T) - sum_{S proper, min T in S} C(S) H(T \ S)         (Eq. 38)                    */
typedef struct {
    int n, nf, absolute;
    const xreal *d;           /* [nf][2^n] */
    const double *sigma;      /* [nf] or NULL (all zero) */
    uint32_t T;
    uint32_t S[MAXF];
    xreal acc;
} o2b_ctx;

static void o2b_rec(o2b_ctx *c, int site, xreal w)
{
    while (site < c->n && !(c->T >> site & 1)) ++site;
    if (site == c->n) {
        int a; xreal p = w;
        for (a = 0; a < c->nf; ++a) p *= c->d[((size_t)a << c->n) + c->S[a]];
        c->acc += p;
        return;
    }
    int a, b;
    uint32_t bit = 1u << site;
    for (a = 0; a < c->nf; ++a) {
        if (c->sigma && c->sigma[a] != 0.0) {         /* one flavour: 2 sigma_a */
            c->S[a] |= bit;
            o2b_rec(c, site + 1, w * (xreal)2 * (xreal)absd(c->sigma[a], c->absolute));
            c->S[a] &= ~bit;
        }
        for (b = a + 1; b < c->nf; ++b) {             /* two flavours a<b: 2 */
            c->S[a] |= bit; c->S[b] |= bit;
            o2b_rec(c, site + 1, w * (xreal)2);
            c->S[a] &= ~bit; c->S[b] &= ~bit;
        }
    }
}

int cos_o2b_polynomial(int n, int nf, const double *A /*[nf][n][n]*/, const double *sigma, int absolute, double *out)
{
    if (n < 1 || n > MAXN || nf < 2 || nf > MAXF) return 1;
    uint32_t full = 1u << n, T;
    xreal *d = (xreal *)malloc(sizeof(xreal) * full * nf);
    xreal *H = (xreal *)malloc(sizeof(xreal) * full);
    xreal *C = (xreal *)malloc(sizeof(xreal) * full);
    if (!d || !H || !C) { free(d); free(H); free(C); return 2; }
    int a;
    for (a = 0; a < nf; ++a)
        for (T = 0; T < full; ++T)
            d[((size_t)a << n) + T] = x_minor_or_perm(n, A + (size_t)a * n * n, T, 0.0, absolute);
    o2b_ctx c;
    memset(&c, 0, sizeof c);
    c.n = n; c.nf = nf; c.d = d; c.sigma = sigma; c.absolute = absolute;
    H[0] = 1;
    for (T = 1; T < full; ++T) {
        c.T = T; c.acc = 0;
        memset(c.S, 0, sizeof c.S);
        o2b_rec(&c, 0, 1);
        H[T] = c.acc;
    }
    if (absolute == 2) cdet_route_scale(n, H, C);
    else cdet_recursion(n, H, C);
    for (T = 1; T < full; ++T) out[T - 1] = (double)C[T];
    free(d); free(H); free(C);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O3: the recurrences as printed, with sparse maps V^(l)[key] (open-addressing hash map).
 * ---------------------------------------------------------------------------------------- */

typedef struct { uint64_t hi, lo; } key128;
typedef struct { key128 *keys; double *vals; uint8_t *used; size_t cap, cnt; } smap;

static int smap_init(smap *m, size_t cap)
{
    m->cap = cap; m->cnt = 0;
    m->keys = (key128 *)malloc(sizeof(key128) * cap);
    m->vals = (double *)malloc(sizeof(double) * cap);
    m->used = (uint8_t *)calloc(cap, 1);
    return (m->keys && m->vals && m->used) ? 0 : 1;
}
static void smap_free(smap *m) { free(m->keys); free(m->vals); free(m->used); m->keys = 0; m->vals = 0; m->used = 0; }
static size_t smap_hash(key128 k, size_t cap)
{
    uint64_t x = k.lo * 0x9E3779B97F4A7C15ull ^ (k.hi + 0x7F4A7C15ull) * 0xC2B2AE3D27D4EB4Full;
    x ^= x >> 29; x *= 0xBF58476D1CE4E5B9ull; x ^= x >> 32;
    return (size_t)(x & (cap - 1));
}
static int smap_add(smap *m, key128 k, double v);
static int smap_grow(smap *m)
{
    smap b; size_t i;
    if (smap_init(&b, m->cap * 2)) return 1;
    for (i = 0; i < m->cap; ++i) if (m->used[i]) smap_add(&b, m->keys[i], m->vals[i]);
    smap_free(m); *m = b;
    return 0;
}
static int smap_add(smap *m, key128 k, double v)       /* V[key] += v */
{
    if ((m->cnt + 1) * 10 > m->cap * 7) if (smap_grow(m)) return 1;
    size_t i = smap_hash(k, m->cap);
    while (m->used[i]) {
        if (m->keys[i].hi == k.hi && m->keys[i].lo == k.lo) { m->vals[i] += v; return 0; }
        i = (i + 1) & (m->cap - 1);
    }
    m->used[i] = 1; m->keys[i] = k; m->vals[i] = v; ++m->cnt;
    return 0;
}

/* ---- Algorithm 3.  Canonical state of Eq. 79-80 ----
 *   qhat = (ubar, vbar, tau_u, lam_u, m, eta),  eta_r = (tau_r, lam_r) if m_r = 1.
 * Key packing: lo = m (2 bits per interaction) | ubar<<24 | vbar<<28 | tau_u<<32 | lam_u<<33;
 *              hi = eta, 4 bits per interaction (bit0 = tau: 1 = shift, bits 1..3 = lam).
 * The function Shift of Alg. 3 maps absolute labels to exactly this record;
 * iterating "w in [N] \ R" over the canonical visited set R_c = {j: m_j>=1} U {j+n: m_j=2}
 * gives two absolute endpoints for m_j = 0 and one for m_j = 1 (Lemma 7).                        */
typedef struct { int u, v, tau_u, lam_u; int m[MAXN]; int eta_tau[MAXN], eta_lam[MAXN]; } a3_state;

static key128 a3_pack(const a3_state *s, int n)
{
    key128 k; int i;
    k.lo = 0; k.hi = 0;
    for (i = 0; i < n; ++i) {
        k.lo |= (uint64_t)s->m[i] << (2 * i);
        if (s->m[i] == 1) k.hi |= (uint64_t)((s->eta_tau[i] & 1) | (s->eta_lam[i] << 1)) << (4 * i);
    }
    k.lo |= (uint64_t)s->u << 24 | (uint64_t)s->v << 28 | (uint64_t)s->tau_u << 32 | (uint64_t)s->lam_u << 33;
    return k;
}
static void a3_unpack(key128 k, int n, a3_state *s)
{
    int i;
    for (i = 0; i < n; ++i) {
        s->m[i] = (int)(k.lo >> (2 * i) & 3);
        int e = (int)(k.hi >> (4 * i) & 15);
        s->eta_tau[i] = e & 1; s->eta_lam[i] = e >> 1;
    }
    s->u = (int)(k.lo >> 24 & 15); s->v = (int)(k.lo >> 28 & 15);
    s->tau_u = (int)(k.lo >> 32 & 1); s->lam_u = (int)(k.lo >> 33 & 7);
}

/* Returns the physical connected sum S_n; *n_states / *n_updates (optional) count map entries
 * and "+=" operations (the CPU baseline's edge visits).  Readings G1-G3 of SURVEY.md 8(c):
 * A_{lambda_n} -> A_{lambda_u}; final loop S += V * (-A) / V * (-sigma); n = 1: S -= sum sigma^2. */
double cos_o3_alg3(int n, int nf, const double *A, const double *sigma_in, int absolute,
                   long long *n_states, long long *n_updates)
{
    if (n < 1 || n > MAXN || nf < 1 || nf > MAXF) return NAN;
    const int N = 2 * n;
    double sigma[MAXF]; int l, layer;
    for (l = 0; l < nf; ++l) sigma[l] = sigma_in ? absd(sigma_in[l], absolute) : 0.0;
    const double minus = absolute ? 1.0 : -1.0;
    long long states = 0, updates = 0;
    smap cur, nxt;
    if (smap_init(&cur, 1024)) return NAN;
    /* initial states, Eq. 66-67: endpoint 1 (index 0), every flavour, normal and shift */
    for (l = 0; l < nf; ++l) {
        int tau;
        for (tau = 0; tau < 2; ++tau) {
            if (tau == 1 && !sigma_in) continue;      /* no counterterm: shift heads carry weight 0 */
            a3_state s; memset(&s, 0, sizeof s);
            s.u = 0; s.v = 0; s.tau_u = tau; s.lam_u = l; s.m[0] = 1; s.eta_tau[0] = tau; s.eta_lam[0] = l;
            smap_add(&cur, a3_pack(&s, n), 1.0);
        }
    }
    for (layer = 0; layer <= N - 2; ++layer) {
        size_t idx;
        if (smap_init(&nxt, cur.cap)) return NAN;
        states += (long long)cur.cnt;
        for (idx = 0; idx < cur.cap; ++idx) {
            if (!cur.used[idx]) continue;
            a3_state s; a3_unpack(cur.keys[idx], n, &s);
            const double om = cur.vals[idx];
            /* Rule 1: continue the cycle (normal head only) */
            if (s.tau_u == 0) {
                int w;
                for (w = 0; w < N; ++w) {
                    int r = w % n;
                    /* visited? canonical R_c: slot r visited iff m_r>=1, slot r+n iff m_r==2 */
                    int visited = (w < n) ? (s.m[r] >= 1) : (s.m[r] == 2);
                    if (visited) continue;
                    a3_state t = s;
                    if (s.m[r] == 1) { t.m[r] = 2; t.eta_tau[r] = 0; t.eta_lam[r] = 0; }   /* partner record removed */
                    else { t.m[r] = 1; t.eta_tau[r] = s.tau_u; t.eta_lam[r] = s.lam_u; }   /* insert (w, tau_u, lam_u) */
                    t.v = r;
                    smap_add(&nxt, a3_pack(&t, n), om * absd(A[(s.lam_u * n + s.v) * n + r], absolute));
                    ++updates;
                }
            }
            /* Rule 2: close the cycle and open the next canonical head */
            {
                double omc = (s.tau_u == 0) ? minus * om * absd(A[(s.lam_u * n + s.v) * n + s.u], absolute)
                                            : minus * om * sigma[s.lam_u];
                int j = -1, i;
                for (i = 0; i < n; ++i) if (s.m[i] == 1) { j = i; break; }
                if (j >= 0) {
                    int tau_p = s.eta_tau[j], lam_p = s.eta_lam[j];
                    a3_state t = s;
                    t.m[j] = 2; t.eta_tau[j] = 0; t.eta_lam[j] = 0; t.u = j; t.v = j;
                    for (l = 0; l < nf; ++l) {
                        if (tau_p == 1 && l != lam_p) continue;           /* Lambda_p, Eq. 71 */
                        t.tau_u = 0; t.lam_u = l;
                        smap_add(&nxt, a3_pack(&t, n), omc); ++updates;
                    }
                    if (sigma_in) {                                       /* shift successor, Eq. 72 */
                        t.tau_u = 1; t.lam_u = lam_p;
                        smap_add(&nxt, a3_pack(&t, n), omc); ++updates;
                    }
                }
            }
        }
        smap_free(&cur); cur = nxt;
    }
    double S = 0.0; size_t idx;
    states += (long long)cur.cnt;
    for (idx = 0; idx < cur.cap; ++idx) {
        if (!cur.used[idx]) continue;
        a3_state s; a3_unpack(cur.keys[idx], n, &s);
        if (s.tau_u == 0) S += cur.vals[idx] * minus * absd(A[(s.lam_u * n + s.v) * n + s.u], absolute);
        else              S += cur.vals[idx] * minus * sigma[s.lam_u];
        ++updates;
    }
    smap_free(&cur);
    if (n == 1 && sigma_in) for (l = 0; l < nf; ++l) S -= sigma[l] * sigma[l] * (absolute ? 0.0 : 1.0);
    if (n_states) *n_states = states;
    if (n_updates) *n_updates = updates;
    return S;
}

/* ---- Uniform SU(N_f) rooted recurrence with all-subset readouts (Eq. 8-15) ----
 * state (r, h, e, m); branch r propagates only through labels j >= r (Eq. 11) with weight
 * (2 - m_j) A_ej; close-and-open at j = min{i >= r : m_i = 1} with factor -N_f A_eh (Eq. 12);
 * readout O_S at layer 2|S|-1 from states with m = 2 1_S (Eq. 13-15).  Initial states
 * (r, r, r, e_r) <- 1 (reading G8).  all_subsets == 0: only r = 0 and out[0] = O_{[n]}.
 * Optional true-diagonal shift (reading G12): with sigma != 0 a singly occupied
 * current interaction may be completed by a counterterm one-cycle, weight -sigma (closing N_f times
 * sigma/N_f), times 2 for the first endpoint (either endpoint of interaction r can be the shift). */
int cos_o3_uniform(int n, int nf, const double *A, double sigma_in, int all_subsets, int absolute,
                   double *out, long long *n_states, long long *n_updates)
{
    if (n < 1 || n > MAXN || nf < 1) return 1;
    const int N = 2 * n;
    const double minus = absolute ? 1.0 : -1.0;
    const double sigma = absd(sigma_in, absolute);
    int n_out = all_subsets ? (1 << n) - 1 : 1, layer, r;
    long long states = 0, updates = 0;
    memset(out, 0, sizeof(double) * n_out);
    smap cur, nxt;
    if (smap_init(&cur, 1024)) return 2;
    for (r = 0; r < (all_subsets ? n : 1); ++r) {
        key128 k; k.hi = 0;
        k.lo = (uint64_t)1 << (2 * r) | (uint64_t)r << 24 | (uint64_t)r << 28 | (uint64_t)r << 32;
        smap_add(&cur, k, 1.0);
    }
    for (layer = 0; layer <= N - 1; ++layer) {
        size_t idx;
        if (smap_init(&nxt, cur.cap)) return 2;
        states += (long long)cur.cnt;
        for (idx = 0; idx < cur.cap; ++idx) {
            if (!cur.used[idx]) continue;
            const uint64_t lo = cur.keys[idx].lo;
            const double om = cur.vals[idx];
            int m[MAXN], i, j;
            for (i = 0; i < n; ++i) m[i] = (int)(lo >> (2 * i) & 3);
            const int h = (int)(lo >> 24 & 15), e = (int)(lo >> 28 & 15);
            r = (int)(lo >> 32 & 15);
            /* continuation, Eq. 11 */
            for (j = r; j < n && layer < N - 1; ++j) {
                if (m[j] >= 2) continue;
                key128 k; k.hi = 0;
                k.lo = (lo & ~((uint64_t)15 << 28)) + ((uint64_t)1 << (2 * j));
                k.lo |= (uint64_t)j << 28;
                smap_add(&nxt, k, om * (double)(2 - m[j]) * absd(A[e * n + j], absolute)); ++updates;
            }
            /* counterterm one-cycle at the partner of the current endpoint (reading G12) */
            if (sigma_in != 0.0 && m[e] == 1 && layer < N - 1) {
                key128 k; k.hi = 0;
                k.lo = lo + ((uint64_t)1 << (2 * e));
                smap_add(&nxt, k, om * minus * sigma * (layer == 0 ? 2.0 : 1.0)); ++updates;
            }
            /* close: -N_f A_eh, then open the canonical next head (Eq. 12) or read out (Eq. 14-15) */
            {
                const double omc = om * minus * (double)nf * absd(A[e * n + h], absolute);
                int jm = -1;
                for (i = r; i < n; ++i) if (m[i] == 1) { jm = i; break; }
                if (jm >= 0) {
                    if (layer < N - 1) {
                        key128 k; k.hi = 0;
                        k.lo = (lo & ~(((uint64_t)15 << 24) | ((uint64_t)15 << 28))) + ((uint64_t)1 << (2 * jm));
                        k.lo |= (uint64_t)jm << 24 | (uint64_t)jm << 28;
                        smap_add(&nxt, k, omc); ++updates;
                    }
                } else {
                    uint32_t S = 0;
                    for (i = 0; i < n; ++i) if (m[i] == 2) S |= 1u << i;
                    if (all_subsets) { out[S - 1] += omc; ++updates; }
                    else if (S == (1u << n) - 1) { out[0] += omc; ++updates; }
                }
            }
        }
        smap_free(&cur); cur = nxt;
    }
    smap_free(&cur);
    if (n_states) *n_states = states;
    if (n_updates) *n_updates = updates;
    return 0;
}
