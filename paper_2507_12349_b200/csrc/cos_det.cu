// cos_det.cu -- the flavour-polynomial (determinant) route of PAPER.md:267-315 on the device, SURVEY.md 8(f).3:
// principal minors d_a(S) (Eq. 34), full moments H(T) through the local tensor L_i (Eq. 35-36) and the connected
// coefficients C(T) by the subset recursion Eq. 38.  An independent second evaluator of what cos_eval computes with
// the all-subset readouts ("providing an independent comparison with SB-CoS for non-uniform matrices and
// shifts"); it shares nothing with the DAG path but the input / output layout.
//
// Precision: the connected value is what is left after Eq. 38 has subtracted every disconnected product of smaller
// moments, which on physical propagators (diagonal ~ -rho, off-diagonal ~ 1e-2) is many orders below H(T) itself
// (|C| / H ~ 1e-8 at n = 6, ~1e-22 at n = 10).  The paper moves this route to double-double arithmetic for that
// reason; every kernel here is a template on the number type: double, or dd = an unevaluated sum
// hi + lo of two doubles (~106 bits, error-free transformations built on FMA).
//
// Lane = configuration everywhere (the configuration index is the contiguous one of every array), so all subset
// loops are warp-uniform and every global access is one coalesced 256-byte line.
#include "cos_kernels.cuh"

namespace cosb {

namespace {

// ---- double-double arithmetic (Dekker / Knuth error-free transformations; two_prod through FMA)
struct dd { double hi, lo; };

__device__ __forceinline__ dd quick_two_sum(double a, double b)       // |a| >= |b|
{
    const double s = __dadd_rn(a, b);
    return {s, __dsub_rn(b, __dsub_rn(s, a))};
}
__device__ __forceinline__ dd two_sum(double a, double b)
{
    const double s = __dadd_rn(a, b), bb = __dsub_rn(s, a);
    return {s, __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb))};
}
__device__ __forceinline__ dd two_prod(double a, double b)
{
    const double p = __dmul_rn(a, b);
    return {p, __fma_rn(a, b, -p)};
}

__device__ __forceinline__ double r_add(double a, double b) { return a + b; }
__device__ __forceinline__ double r_mul(double a, double b) { return a * b; }
__device__ __forceinline__ double r_muld(double a, double b) { return a * b; }
__device__ __forceinline__ double r_div(double a, double b) { return a / b; }
__device__ __forceinline__ double r_neg(double a) { return -a; }
__device__ __forceinline__ double r_hi(double a) { return a; }
__device__ __forceinline__ double r_round(double a) { return a; }
__device__ __forceinline__ double r_fma(double a, double b, double acc) { return fma(a, b, acc); }
__device__ __forceinline__ double r_scale2(double a, int e) { return ldexp(a, e); }

// Addition with the low parts added in plain fp64 (11 operations instead of 20): the error is bounded by
// ~2^-104 (|a| + |b|), not by 2^-104 |a + b| -- exactly the kind of bound this route needs, since its tolerance is
// relative to the sum of absolute values R anyway (include/cos.h).
__device__ __forceinline__ dd r_add(dd a, dd b)
{
    const dd s = two_sum(a.hi, b.hi);
    return quick_two_sum(s.hi, __dadd_rn(s.lo, __dadd_rn(a.lo, b.lo)));
}
__device__ __forceinline__ dd r_mul(dd a, dd b)
{
    const dd p = two_prod(a.hi, b.hi);
    return quick_two_sum(p.hi, __dadd_rn(p.lo, __fma_rn(a.hi, b.lo, __dmul_rn(a.lo, b.hi))));
}
__device__ __forceinline__ dd r_muld(dd a, double b)
{
    const dd p = two_prod(a.hi, b);
    return quick_two_sum(p.hi, __fma_rn(a.lo, b, p.lo));
}
__device__ __forceinline__ dd r_neg(dd a) { return {-a.hi, -a.lo}; }
__device__ __forceinline__ dd r_div(dd a, dd b)
{
    const double q1 = a.hi / b.hi;
    dd r = r_add(a, r_neg(r_muld(b, q1)));
    const double q2 = r.hi / b.hi;
    r = r_add(r, r_neg(r_muld(b, q2)));
    const double q3 = r.hi / b.hi;
    return r_add(quick_two_sum(q1, q2), dd{q3, 0.0});
}
__device__ __forceinline__ double r_hi(dd a) { return a.hi; }
__device__ __forceinline__ double r_round(dd a) { return __dadd_rn(a.hi, a.lo); }
__device__ __forceinline__ dd r_fma(dd a, dd b, dd acc) { return r_add(acc, r_mul(a, b)); }
__device__ __forceinline__ dd r_scale2(dd a, int e) { return {ldexp(a.hi, e), ldexp(a.lo, e)}; }   // exact

template <class R> __device__ __forceinline__ R r_from(double x);
template <> __device__ __forceinline__ double r_from<double>(double x) { return x; }
template <> __device__ __forceinline__ dd r_from<dd>(double x) { return {x, 0.0}; }

// element e of an array of R that starts at p (dd elements are 16-byte {hi, lo} pairs: one LDG.128 / STG.128)
__device__ __forceinline__ double r_load(const double* p, size_t e) { return p[e]; }
__device__ __forceinline__ void r_store(double* p, size_t e, double v) { p[e] = v; }
__device__ __forceinline__ dd r_load(const dd* p, size_t e)
{
    const double2 v = reinterpret_cast<const double2*>(p)[e];
    return {v.x, v.y};
}
__device__ __forceinline__ void r_store(dd* p, size_t e, dd v) { reinterpret_cast<double2*>(p)[e] = make_double2(v.hi, v.lo); }

__device__ __forceinline__ uint32_t deposit_bits(uint32_t k, uint32_t mask)
{
    // the k-th submask of `mask`: bit i of k goes to the position of the i-th set bit of mask
    uint32_t r = 0;
    while (mask) {
        const uint32_t low = mask & (0u - mask);
        if (k & 1u) r |= low;
        k >>= 1;
        mask ^= low;
    }
    return r;
}

__device__ __forceinline__ size_t wide_mul(uint32_t x, uint32_t y)      // 32 x 32 -> 64 bits, one instruction
{
    unsigned long long r;
    asm("mul.wide.u32 %0, %1, %2;" : "=l"(r) : "r"(x), "r"(y));
    return (size_t)r;
}

__device__ __forceinline__ uint32_t binom_u32(int p, int r)
{
    if (r < 0 || r > p) return 0;
    uint32_t b = 1;
    for (int j = 1; j <= r; ++j) b = b * (uint32_t)(p - r + j) / (uint32_t)j;   // exact at every step
    return b;
}

}  // namespace

// order[rank] = subset T, ranks sorted by decreasing |T| (colex inside one size): the expensive subsets of the
// moment kernel are scheduled first, and the recursion kernel walks the sizes from the back.
__global__ void cos_det_order_kernel(int n, uint32_t* order)
{
    const uint32_t T = blockIdx.x * blockDim.x + threadIdx.x;
    if (T >= (1u << n)) return;
    const int k = __popc(T);
    uint32_t rank = 0;
    for (int j = k + 1; j <= n; ++j) rank += binom_u32(n, j);
    uint32_t m = T;
    for (int i = 1; m; ++i) {
        const int p = __ffs(m) - 1;
        rank += binom_u32(p, i);
        m &= m - 1;
    }
    order[rank] = T;
}

// Eq. 34: d_blk(S) = det A^{(blk)}[S, S] for every S (d(empty) = 1).  One thread per (configuration, S, block):
// the |S| x |S| principal sub-block is gathered into local memory and eliminated with partial pivoting.
template <class R>
__global__ void __launch_bounds__(128) cos_det_minors_kernel(const DetArgs a)
{
    const int n = a.n;
    const long long c = (long long)blockIdx.x * 32 + threadIdx.x;
    const uint32_t idx = blockIdx.y * blockDim.y + threadIdx.y;          // blk * 2^n + S
    if (c >= a.batch || idx >= ((uint32_t)a.n_blocks << n)) return;
    const uint32_t S = idx & ((1u << n) - 1u);
    const int blk = (int)(idx >> n);
    int v[COS_DET_MAX_N];
    int k = 0;
    for (int i = 0; i < n; ++i)
        if (S >> i & 1u) v[k++] = i;
    R M[COS_DET_MAX_N * COS_DET_MAX_N];
    // endpoint of vertex i under the current sublattice assignment: i * n_sub + s_i (include/cos.h); d = n * n_sub
    const int d = n * a.nsub;
    if (a.nsub == 2)
        for (int r = 0; r < k; ++r) v[r] = 2 * v[r] + (int)(a.assign >> v[r] & 1u);
    const double* A = a.G + (size_t)blk * d * d * a.batch + c;
    for (int r = 0; r < k; ++r)
        for (int q = 0; q < k; ++q) M[r * k + q] = r_from<R>(A[(size_t)(v[r] * d + v[q]) * a.batch]);
    R det = r_from<R>(1.0);
    for (int p = 0; p < k; ++p) {
        int piv = p;
        double best = fabs(r_hi(M[p * k + p]));
        for (int r = p + 1; r < k; ++r) {
            const double x = fabs(r_hi(M[r * k + p]));
            if (x > best) { best = x; piv = r; }
        }
        if (best == 0.0) { det = r_from<R>(0.0); break; }
        if (piv != p) {
            for (int q = p; q < k; ++q) {
                const R t = M[p * k + q];
                M[p * k + q] = M[piv * k + q];
                M[piv * k + q] = t;
            }
            det = r_neg(det);
        }
        const R pv = M[p * k + p];
        det = r_mul(det, pv);
        for (int r = p + 1; r < k; ++r) {
            const R f = r_neg(r_div(M[r * k + p], pv));
            for (int q = p + 1; q < k; ++q) M[r * k + q] = r_fma(f, M[p * k + q], M[r * k + q]);
        }
    }
    r_store((R*)a.minors, (size_t)idx * a.batch + c, det);
}

// Eq. 35-36: H(T) = sum over the occupations of the sites of T -- a pair of flavours {a < b} (weight 2) or one flavour a
// with its counterterm (weight 2 sigma_a); no flavour means "not in T", three flavours weigh 0 -- of
// prod_a d_a(S_a), S_a = sites occupied by flavour a.  Flavours are called 0, 1, 2; with two flavours (THREE = false)
// the middle one is absent (S_1 = empty), which leaves exactly the occupations {02}, {0}, {2}.
//
// CTA = (subset T, batch tile); its warps split the 2^|T| choices of S_0 (3^|T| terms each, so the split is even)
// and their partial sums are added in warp order (deterministic).  Loop nest for one S_0, U = T \ S_0:
//   X subset of S_0  : sites of the pair {01};   the rest F_0 = S_0 \ X is {02} or {0}
//   Y subset of U    : sites of S_1 outside S_0 ({12} or {1});   the rest U \ Y is {2}
//   R_0 subset of F_0, R_1 subset of Y : the sites that take the pair with flavour 2; the others pay sigma_0 / sigma_1
// term = d_0(S_0) d_1(X + Y) d_2((U \ Y) + R_0 + R_1) sigma_2^|U \ Y| sigma_0^|F_0 \ R_0| sigma_1^|Y \ R_1|, times 2^|T|.
// The weights (powers of the caller's fp64 sigma, in the working precision, tabulated in shared memory) depend only on
// set sizes and are the same for every configuration; sigma_a = 0 removes the "single a" choice from the loops, and
// sigma_1 = 0 lets the sums over d_1 and d_2 factorise.
template <class R, bool THREE>
__global__ void __launch_bounds__(256) cos_det_moment_kernel(const DetArgs a)
{
    __shared__ R pw2[COS_DET_MAX_N + 1];                              // sigma_2^k
    __shared__ R pw01[COS_DET_MAX_N + 1][COS_DET_MAX_N + 1];          // sigma_0^k0 sigma_1^k1
    __shared__ R red[8][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (threadIdx.x < (COS_DET_MAX_N + 1) * (COS_DET_MAX_N + 1)) {
        const int k0 = threadIdx.x / (COS_DET_MAX_N + 1), k1 = threadIdx.x % (COS_DET_MAX_N + 1);
        R p = r_from<R>(1.0), q = r_from<R>(1.0);
        for (int i = 0; i < k0; ++i) p = r_muld(p, a.sigma[0]);
        for (int i = 0; i < k1; ++i) p = r_muld(p, a.sigma[1]);
        for (int i = 0; i < k1; ++i) q = r_muld(q, a.sigma[2]);
        pw01[k0][k1] = p;
        if (k0 == 0) pw2[k1] = q;
    }
    __syncthreads();
    const uint32_t n_T = (1u << a.n) - 1u;                   // blockIdx.x = tile * n_T + rank: a tile's subsets are neighbours
    const uint32_t T = a.order[blockIdx.x % n_T];
    long long c = (long long)(blockIdx.x / n_T) * 32 + lane;
    const bool valid = c < a.batch;
    if (!valid) c = a.batch - 1;
    const uint32_t B = (uint32_t)a.batch;                    // < 2^31 (checked by the C-ABI): subset x B is one IMAD.WIDE
    const R* m0 = (const R*)a.minors + (size_t)((uint32_t)a.blk[0] << a.n) * B + c;
    const R* m1 = (const R*)a.minors + (size_t)((uint32_t)a.blk[1] << a.n) * B + c;
    const R* m2 = (const R*)a.minors + (size_t)((uint32_t)a.blk[2] << a.n) * B + c;
    const int kT = __popc(T);
    // sigma_f = 0: no site may pay that counterterm, so the sites of that class are forced into the pair with flavour 2
    // (sigma_0, sigma_1) or Y must be all of U (sigma_2)
    const bool z0 = a.sigma[0] == 0.0, z1 = a.sigma[1] == 0.0, z2 = a.sigma[2] == 0.0;
    R acc = r_from<R>(0.0);
    // The 2^|T| choices of S_0 are split over the 8 warps.  A choice costs ~3^|S_0| + 2^|T| terms, so a plain stride (warp
    // = the three low bits of k) would hand warp 7 the choices with three more sites than warp 0's (27 x the work) and
    // leave the others at the final barrier (max / mean load 2.19): the low bits are w XOR a hash of the high part instead,
    // so that every warp meets every low-bit pattern equally often whatever the weight of the high part -- static (the
    // summation order stays fixed), max / mean load 1.17 at |T| = 10, 1.29 at |T| = 8.
    for (uint32_t i = 0; (i << 3) < (1u << kT) || i == 0; ++i) {
        const uint32_t k = (kT >= 3) ? ((i << 3) | (((uint32_t)w ^ i ^ (i >> 3) ^ (i >> 6)) & 7u)) : (uint32_t)w;
        if (k >= (1u << kT)) break;
        const uint32_t S0 = deposit_bits(k, T), U = T & ~S0;
        R accS0 = r_from<R>(0.0);
        for (uint32_t X = THREE ? S0 : 0u;; X = (X - 1) & S0) {
            const uint32_t F0 = S0 & ~X;
            // inner_sum(fixed, fr0, fr1) = sum over R subset of (fr0 | fr1) of sigma_0^|fr0 \ R| sigma_1^|fr1 \ R| d_2(fixed | R):
            // the sites of fr0 (in F0) and fr1 (in Y) choose "pair with flavour 2" (in R) or "single" (weight sigma_0 /
            // sigma_1); one sub-mask loop over both classes
            auto inner_sum = [&](const uint32_t fixed, const uint32_t fr0, const uint32_t fr1) -> R {
                const uint32_t free_ = fr0 | fr1;
                const R* p2 = m2 + wide_mul(fixed, B);
                R inner = r_from<R>(0.0);
                if (__popc(free_) < 2) {
                    for (uint32_t Rr = free_;; Rr = (Rr - 1) & free_) {
                        inner = r_fma(pw01[__popc(fr0 & ~Rr)][__popc(fr1 & ~Rr)], r_load(p2, wide_mul(Rr, B)), inner);
                        if (Rr == 0u) break;
                    }
                } else {
                    // four sub-masks per iteration (the two lowest free sites in / out): four independent look-ups
                    // in flight instead of one dependent load per term
                    const uint32_t b0 = free_ & (0u - free_), f1 = free_ ^ b0, b1 = f1 & (0u - f1), rest = f1 ^ b1;
                    const int a0 = (b0 & fr0) ? 1 : 0, a1 = (b1 & fr0) ? 1 : 0;     // class of b0 / b1: 1 = F0, 0 = Y
                    for (uint32_t Rh = rest;; Rh = (Rh - 1) & rest) {
                        const int k0 = __popc(fr0 & rest & ~Rh), k1 = __popc(fr1 & rest & ~Rh);
                        const R* q = p2 + wide_mul(Rh, B);
                        const R v11 = r_load(q, wide_mul(b0 | b1, B)), v01 = r_load(q, wide_mul(b1, B));
                        const R v10 = r_load(q, wide_mul(b0, B)), v00 = r_load(q, 0);
                        inner = r_fma(pw01[k0][k1], v11, inner);
                        inner = r_fma(pw01[k0 + a0][k1 + 1 - a0], v01, inner);                  // b0 single
                        inner = r_fma(pw01[k0 + a1][k1 + 1 - a1], v10, inner);                  // b1 single
                        inner = r_fma(pw01[k0 + a0 + a1][k1 + 2 - a0 - a1], v00, inner);        // both single
                        if (Rh == 0u) break;
                    }
                }
                return inner;
            };
            const uint32_t fr0 = z0 ? 0u : F0;
            if (THREE && z1) {
                // sigma_1 = 0: every site of Y pairs with flavour 2, so d_2 is taken at U | (forced part of F0) | R for every
                // Y: the d_2 sum and the d_1 sum over Y factorise (2^|F0| + 2^|U| terms instead of their product)
                const R inner = inner_sum(U | (F0 & ~fr0), fr0, 0u);
                R sumY = r_from<R>(0.0);
                for (uint32_t Y = U;; Y = (Y - 1) & U) {
                    const R w2 = pw2[__popc(U & ~Y)];
                    if (r_hi(w2) != 0.0) sumY = r_fma(w2, r_load(m1, wide_mul(X | Y, B)), sumY);
                    if (Y == 0u || z2) break;
                }
                accS0 = r_fma(inner, sumY, accS0);
            } else {
                for (uint32_t Y = THREE ? U : 0u;; Y = (Y - 1) & U) {
                    const uint32_t base = U & ~Y;
                    const R w2 = pw2[__popc(base)];
                    if (r_hi(w2) != 0.0) {
                        const uint32_t fr1 = z1 ? 0u : Y;
                        R inner = inner_sum(base | ((F0 | Y) & ~(fr0 | fr1)), fr0, fr1);
                        if (THREE) inner = r_mul(inner, r_load(m1, wide_mul(X | Y, B)));
                        accS0 = r_fma(w2, inner, accS0);
                    }
                    if (Y == 0u || (z2 && THREE)) break;
                }
            }
            if (X == 0u) break;
        }
        acc = r_fma(r_load(m0, wide_mul(S0, B)), accS0, acc);
    }
    red[w][lane] = acc;
    __syncthreads();
    if (w == 0 && valid) {
        R s = red[0][lane];
#pragma unroll
        for (int i = 1; i < 8; ++i) s = r_add(s, red[i][lane]);
        // honeycomb: H^{(s)}(T) depends only on the labels of the sites of T, and all 2^n assignments are walked, so every
        // value is met 2^(n - |T|) times: the exact power of two is divided out here (Eq. 54-55)
        s = r_scale2(s, a.nsub == 2 ? 2 * kT - a.n : kT);
        if (a.accumulate) s = r_add(s, r_load((const R*)a.H, wide_mul(T, B) + c));
        r_store((R*)a.H, wide_mul(T, B) + c, s);
    }
}

// Eq. 38: C(T) = H(T) - sum_{S proper subset of T, min T in S} C(S) H(T \ S), sizes in increasing order.  One CTA per
// batch tile; the subsets of one size are independent and are split over the warps.  C is kept in the working
// precision in the workspace (row bitmask(T)) and rounded to fp64 into the caller's output, row bitmask(T) - 1.
template <class R>
__global__ void __launch_bounds__(256) cos_det_connected_kernel(const DetArgs a)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    long long c = (long long)blockIdx.x * 32 + lane;
    const bool valid = c < a.batch;
    if (!valid) c = a.batch - 1;
    const size_t B = (size_t)a.batch;
    const R* H = (const R*)a.H + c;
    R* C = (R*)a.C + c;
    for (int k = 1; k <= a.n; ++k) {
        for (uint32_t i = a.level_off[k] + w; i < a.level_off[k - 1]; i += 8) {
            const uint32_t T = a.order[i];
            const uint32_t r = T & (0u - T), rest = T ^ r;
            R val = r_load(H, (size_t)T * B);
            if (rest) {
                for (uint32_t Q = (rest - 1) & rest;; Q = (Q - 1) & rest) {
                    val = r_fma(r_neg(r_load(C, (size_t)(r | Q) * B)), r_load(H, (size_t)(rest & ~Q) * B), val);
                    if (Q == 0u) break;
                }
            }
            if (valid) {
                r_store(C, (size_t)T * B, val);
                a.out[(size_t)(T - 1u) * B + c] = r_round(val);
            }
        }
        __syncthreads();
    }
}

template <class R>
static cudaError_t launch_det_route_t(const DetArgs& a, cudaStream_t stream)
{
    const uint32_t n_sub = 1u << a.n;
    const uint32_t tiles = (uint32_t)((a.batch + 31) / 32);
    cos_det_order_kernel<<<(n_sub + 255) / 256, 256, 0, stream>>>(a.n, a.order);
    const uint32_t n_minors = (uint32_t)a.n_blocks << a.n;
    // honeycomb (Eq. 54-55): the moments are summed over the sublattice labels of the vertices before Eq. 38 (the
    // connected part of the summed moments is the sum of the connected parts: labels factorise over components)
    DetArgs b = a;
    for (uint32_t assign = 0; assign < (a.nsub == 2 ? n_sub : 1u); ++assign) {
        b.assign = assign;
        b.accumulate = assign > 0;
        cos_det_minors_kernel<R><<<dim3(tiles, (n_minors + 3) / 4), dim3(32, 4), 0, stream>>>(b);
        if (a.three)
            cos_det_moment_kernel<R, true><<<(n_sub - 1) * tiles, 256, 0, stream>>>(b);
        else
            cos_det_moment_kernel<R, false><<<(n_sub - 1) * tiles, 256, 0, stream>>>(b);
    }
    cos_det_connected_kernel<R><<<tiles, 256, 0, stream>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_det_route(const DetArgs& a, cudaStream_t stream)
{
    return a.dd ? launch_det_route_t<dd>(a, stream) : launch_det_route_t<double>(a, stream);
}

}  // namespace cosb
