// cos_kernels.cu -- sm_100a kernels of the CoS / SB-CoS DAG evaluator.
//
//  cos_layer_kernel   north_star (3)+(4): one layer step x_t += c_e L[x_s] (Eq. 16) for every
//                     state of the next layer, plus the terminal readouts of this layer (Eq. 14-15).
//  cos_fused_kernel   the same for small DAGs: every layer in one launch.
//  cos_tabulate_kernel north_star (2): propagator lookup with linear tau-interpolation (Eq. 32).
//  cos_fill_kernel    layer-0 initial states <- 1 (Eq. 66).
//  fp64 FMA peak probe for the roofline report.
//
// Work decomposition of the layer kernel:
//   lane  = configuration (32 per batch tile, the contiguous dimension of every array),
//   warp  = one occupancy-mask block at a time: all group records of the block,
//   CTA   = `masks_per_cta` blocks x one batch tile; the tile's propagator table G (all blocks, d x d,
//           32 configurations) is staged once in shared memory.
// A group record is up to 4 rows (heads) of one colour of the block.  The continuation factor G_lambda[e][j] does not
// depend on the head, so the record is a small product  Y[head][j] = sum_e X[head][e] * G_lambda[e][j]  per
// configuration: for every source endpoint e the TJ factors are loaded ONCE from shared memory and applied to the TH
// source values (factor-application sharing, Eq. 29-31), TH x TJ accumulators live in registers, and every
// source state is read from HBM exactly once, just in time (one step ahead).  Every destination state is written exactly
// once: no atomics, no second pass, HBM traffic = one read + one write per state.
#include "cos_kernels.cuh"
#include "cos_compile.h"

// source-value stages (prefetch depth) of the three register tiles
#ifndef COS_BULK_PREFETCH
#define COS_BULK_PREFETCH 1
#endif
#ifndef COS_L1_AHEAD
#define COS_L1_AHEAD 2
#endif
#ifndef COS_STAGES_A
#define COS_STAGES_A 2
#endif
#ifndef COS_STAGES_B
#define COS_STAGES_B 3
#endif
#ifndef COS_STAGES_C
#define COS_STAGES_C 4
#endif

namespace cosb {

static const int MAX_WARPS = 16;         // 128 registers per thread

__device__ __forceinline__ double lds64(uint32_t addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
// one bulk (TMA) prefetch of a contiguous range into L2; bytes is a multiple of 16
__device__ __forceinline__ void prefetch_l2_bulk(const void* p, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
// asynchronous 8-byte global -> shared copy (LDGSTS): no register staging, completion by commit / wait groups
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
// 16-byte variant (L2 only): program records -> the warp's record slots
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ uint4 lds128u(uint32_t addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint2 lds64u(uint32_t addr)
{
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// What a warp needs to walk the records of one batch tile.
struct TileCtx {
    const char* Xl;                      // source slab of the tile + lane * 8
    char* Yl;                            // destination slab of the tile + lane * 8
    uint32_t gs_lane;                    // shared-memory byte address of Gs[0][lane]
    uint32_t gd_lane;                    // ... of the plain diagonal Gd[0][lane]
    uint32_t d, dstride;                 // table dimension, d * 256 bytes (one table row of 32 configurations)
    uint32_t S_src;                      // states of the source layer
    int prefetch;                        // L2 look-ahead (0: off; else the states fetched ahead when a block is claimed)
    int lane;
};

// Keeps a loop-invariant value in a register: the compiler may not rematerialise it inside the loops below.
__device__ __forceinline__ void pin(uint32_t& v) { asm volatile("" : "+r"(v)); }

// The source values of endpoint e (bit = 1 << e; bit = 0: none) for the heads of a record, 0 where a head has no such state.
template <int THM, bool FUSED>
__device__ __forceinline__ void load_x(const uint32_t bit, double (&x)[THM], uint32_t (&idx)[THM], const uint32_t (&al)[THM],
                                       const char* __restrict__ Xl)
{
#pragma unroll
    for (int t = 0; t < THM; ++t) {
        x[t] = 0.0;
        if (al[t] & bit) {
            const double* p = (const double*)(Xl + ((size_t)idx[t] << 8));
            x[t] = FUSED ? __ldcg(p) : __ldcs(p);
#if COS_L1_AHEAD > 0
            // pull the line this head reads COS_L1_AHEAD states later into L1 (no register needed; the slab is padded)
            if (!FUSED) asm volatile("prefetch.global.L1 [%0+%1];" ::"l"(p), "n"(COS_L1_AHEAD * 256));
#endif
            ++idx[t];
        }
    }
}

// One group record (cos_compile.h) with exactly TJ destination endpoints on a register tile of THM heads (the record's
// TH <= THM heads are a run-time value; unused rows carry x = 0):
//   for every source endpoint e (increasing): TJ factor loads G_lambda[e][j] (shared by the heads), THM x TJ FMAs, and per
//   head the cycle-closing factor G_lambda[e][h] (Eq. 12, 15), which never carries the counterterm (plain diagonal Gd
//   when e == h); then one store per live (head, endpoint).
// The source values stream through D register stages: the loads of endpoint k + D - 1 are in flight while endpoint k is
// applied (stages are named statically -- a register move from a pending load would wait for it).
template <int THM, int TJ, int D, bool FUSED>
__device__ __forceinline__ void group_run(const uint32_t rec, const uint4 q0, const int TH, uint32_t (&idx)[THM],
                                          const uint32_t (&al)[THM], const uint32_t (&hoff)[THM], const TileCtx& c,
                                          double& close)
{
    constexpr int TJ1 = TJ > 0 ? TJ : 1;
    const uint32_t lam = (q0.x >> 8) & 3u;
    const bool do_close = (q0.x >> 10) & 1u;
    uint32_t dstride = c.dstride;
    pin(dstride);
    // shared-memory byte addresses: column j of table row 0 of this colour (+ e * dstride = G_lambda[e][j]), the
    // closing column of every head, and its plain-diagonal entry Gd_lambda[h]
    uint32_t colq[TJ1];
    uint32_t row0 = c.gs_lane + lam * c.d * dstride, gdl = c.gd_lane + ((lam * c.d) << 8);
    pin(row0); pin(gdl);
    {
        uint32_t jm = q0.z;
#pragma unroll
        for (int q = 0; q < TJ; ++q) { colq[q] = row0 + ((uint32_t)(__ffs((int)jm) - 1) << 8); jm &= jm - 1u; pin(colq[q]); }
    }
    double acc[THM][TJ1];
#pragma unroll
    for (int t = 0; t < THM; ++t)
#pragma unroll
        for (int q = 0; q < TJ1; ++q) acc[t][q] = 0.0;
    double cl = 0.0;

    uint32_t em = q0.y;
    uint32_t bq[D];
    double xs[D][THM];
#pragma unroll
    for (int s = 0; s < D; ++s) {
        bq[s] = em & (0u - em);                        // 0 after the last endpoint: load_x then loads nothing
        em ^= bq[s];
        load_x<THM, FUSED>(bq[s], xs[s], idx, al, c.Xl);
    }
    bool live = true;
    while (live) {
#pragma unroll
        for (int s = 0; s < D; ++s) {
            if (live) {
                const uint32_t e = 31u - (uint32_t)__clz((int)bq[s]);
                const uint32_t ro = e * dstride;
                double g[TJ1];
#pragma unroll
                for (int q = 0; q < TJ; ++q) g[q] = lds64(colq[q] + ro);
#pragma unroll
                for (int q = 0; q < TJ; ++q)
#pragma unroll
                    for (int t = 0; t < THM; ++t) acc[t][q] = fma(g[q], xs[s][t], acc[t][q]);
                if (do_close) {      // a head without this source state has x = 0: its (valid) factor load is harmless
#pragma unroll
                    for (int t = 0; t < THM; ++t)
                        cl = fma(lds64(hoff[t] + ((hoff[t] == (e << 8)) ? gdl : row0 + ro)), xs[s][t], cl);
                }
                bq[s] = em & (0u - em);
                em ^= bq[s];
                load_x<THM, FUSED>(bq[s], xs[s], idx, al, c.Xl);
                live = bq[(s + 1) % D] != 0u;
            }
        }
    }
    if (TJ > 0) {
        const uint32_t dw = rec + 16u * (uint32_t)(1 + TH);
        constexpr int ROW2 = (TJ + 1) / 2;          // uint2 per destination row
#pragma unroll
        for (int t = 0; t < THM; ++t) {
            if (t < TH) {
#pragma unroll
                for (int i = 0; i < ROW2; ++i) {
                    const uint2 w2 = lds64u(dw + 8u * (uint32_t)(t * ROW2 + i));
#pragma unroll
                    for (int k = 0; k < 2; ++k) {
                        if (2 * i + k < TJ) {
                            const uint32_t w = k == 0 ? w2.x : w2.y;
                            if (w != DIDX_DEAD) {
                                double* y = (double*)(c.Yl + ((size_t)w << 8));
                                if (FUSED) *y = acc[t][2 * i + k]; else __stcs(y, acc[t][2 * i + k]);
                            }
                        }
                    }
                }
            }
        }
    }
    if (do_close) close += cl;
}

// Dispatch of a record on its register tile (THM heads, up to TJM endpoints, D source stages).
template <int THM, int TJM, int D, bool FUSED>
__device__ __forceinline__ void group_tile(const uint32_t rec, const uint4 q0, const TileCtx& c, double& close)
{
    const int TH = (int)(q0.x & 7u), TJ = (int)((q0.x >> 3) & 31u);
    uint32_t idx[THM], al[THM], hoff[THM];
#pragma unroll
    for (int t = 0; t < THM; ++t) {
        idx[t] = 0u; al[t] = 0u; hoff[t] = 0u;
        if (t < TH) {
            const uint4 qh = lds128u(rec + 16u * (uint32_t)(1 + t));
            idx[t] = qh.x; al[t] = qh.y; hoff[t] = qh.z << 8;
            // L2 look-ahead: the sources of the record GROUP_LOOKAHEAD records later (contiguous: one bulk prefetch)
            if (t == 0 && c.prefetch > 0 && c.lane == 0) {
                const uint32_t ahead2 = (q0.x >> 18) & 0x3Fu;
                if (ahead2) prefetch_l2_bulk(c.Xl + ((size_t)qh.w << 8), ahead2 << 9);
            }
        }
    }
#define COS_RUN_CASE(TJ_) \
    case TJ_: group_run<THM, (TJ_ <= TJM ? TJ_ : 0), D, FUSED>(rec, q0, TH, idx, al, hoff, c, close); break;
    switch (TJ) {
        COS_RUN_CASE(0) COS_RUN_CASE(1) COS_RUN_CASE(2) COS_RUN_CASE(3) COS_RUN_CASE(4) COS_RUN_CASE(5) COS_RUN_CASE(6)
        default:
            if (TJM > 6) {
                switch (TJ) {
                    COS_RUN_CASE(7) COS_RUN_CASE(8)
                    default:
                        if (TJM > 8) {
                            switch (TJ) {
                                COS_RUN_CASE(9) COS_RUN_CASE(10) COS_RUN_CASE(11) COS_RUN_CASE(12)
                                default: break;
                            }
                        }
                        break;
                }
            }
            break;
    }
#undef COS_RUN_CASE
}

// All source blocks [m_begin, m_end) of one layer for one batch tile: the body shared by the per-layer kernel and the
// fused small-DAG kernel.  s_next (shared) must be 0 and visible to the CTA on entry.
template <bool FUSED>
__device__ __forceinline__ void layer_blocks(const LayerArgs& a, const uint32_t m_begin, const uint32_t m_end,
                                             const uint32_t tile, unsigned int& s_next, const uint32_t gs_lane,
                                             const uint32_t rs_warp, const int lane, const bool valid, const long long b)
{
    TileCtx c;
    c.Xl = (const char*)(a.X + (size_t)tile * a.S_src * TILE + lane);
    c.Yl = (char*)(a.Y + (size_t)tile * a.S_dst * TILE + lane);
    c.gs_lane = gs_lane; c.gd_lane = gs_lane + (uint32_t)a.n_slots * (TILE * 8u);
    pin(c.gs_lane); pin(c.gd_lane);
    c.d = (uint32_t)a.d; c.dstride = (uint32_t)a.d * (TILE * 8u);
    c.S_src = a.S_src; c.prefetch = a.prefetch; c.lane = lane;
    const uint2* mtab = (const uint2*)a.mask_off;

    // Blocks are handed to warps dynamically (block sizes vary).  A warp always knows its current AND its next block.
    // The program is read through per-warp shared-memory slots of 256 bytes filled by asynchronous copies one step ahead
    // (lanes 0..15 copy 16 bytes each): slots 0/1 take a block header together with the block's first record, slots 2/3
    // the following records, so that no record field is ever waited for at global-memory latency.
    const uint32_t slot_lane = rs_warp + (uint32_t)(lane & 15) * 16u;
    uint32_t mi = 0;
    if (lane == 0) mi = atomicAdd(&s_next, 1u);
    mi = __shfl_sync(0xFFFFFFFFu, mi, 0) + m_begin;
    const uint4* bp = nullptr;
    uint32_t pb = 0u;                        // block slot of the current block
    if (mi < m_end) {
        bp = (const uint4*)(a.words + __ldg(&mtab[mi]).x);
        if (lane < 16) cp_async16(slot_lane, bp + lane);
    }
    cp_async_commit();
    while (mi < m_end) {
        uint32_t mi_n = 0;
        if (lane == 0) mi_n = atomicAdd(&s_next, 1u);
        mi_n = __shfl_sync(0xFFFFFFFFu, mi_n, 0) + m_begin;
        const uint4* bp_n = nullptr;
        if (mi_n < m_end) {
            const uint2 mt = __ldg(&mtab[mi_n]);
            bp_n = (const uint4*)(a.words + mt.x);
            if (lane < 16) cp_async16(slot_lane + ((pb ^ 1u) << 8), bp_n + lane);
            // L2 look-ahead: the first states of the block this warp takes next (one bulk prefetch, a block away in time)
            if (a.prefetch > 0 && lane == 0) {
                uint32_t cnt = __ldg(&mtab[mi_n + 1].y) - mt.y;
                if (cnt > (uint32_t)a.prefetch) cnt = (uint32_t)a.prefetch;
                if (cnt) prefetch_l2_bulk(c.Xl + ((size_t)mt.y << 8), cnt << 8);
            }
        }
        cp_async_commit();
        cp_async_wait<1>();                  // everything but the copy just issued: the current block's slot is complete
        __syncwarp();
        const uint32_t bs = rs_warp + (pb << 8);
        const uint4 h0 = lds128u(bs);
        const int n_groups = (int)(h0.x & 0xFFFFu);
        const uint32_t flags = h0.x >> 24;
        double close = 0.0;

        const uint4* rec_g = bp + 2;         // global address of the current record
        uint32_t rec = bs + 32u;             // its shared-memory copy
        for (int g = 0; g < n_groups; ++g) {
            const uint4 q0 = lds128u(rec);
            rec_g += q0.x >> 24;
            const uint32_t rec_n = rs_warp + 512u + (((uint32_t)g & 1u) << 8);
            if (g + 1 < n_groups && lane < 16) cp_async16(rec_n + (uint32_t)lane * 16u, rec_g + lane);
            cp_async_commit();
            {   // register tile by head count (cos_compile.h): A = 4 x 6, B = 2 x 8, C = 1 x 12
                const uint32_t th = q0.x & 7u;
                if (th >= 3u) group_tile<TILE_A_HEADS, TILE_A_COLS, COS_STAGES_A, FUSED>(rec, q0, c, close);
                else if (th == 2u) group_tile<TILE_B_HEADS, TILE_B_COLS, COS_STAGES_B, FUSED>(rec, q0, c, close);
                else group_tile<1, GROUP_MAX_COLS, COS_STAGES_C, FUSED>(rec, q0, c, close);
            }
            cp_async_wait<0>();
            __syncwarp();
            rec = rec_n;
        }
        if (flags & FLAG_FRESH) {            // close-and-open: fresh head of every colour (Eq. 12, 70-71)
            // h0.w bit k: a row of this block has already stored its continuation into the fresh-head state of colour k
            // (the coalesced E2/E4 pair): add the closing sum to it
            const uint4 fd = lds128u(bs + 16u);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t didx = k == 0 ? fd.x : k == 1 ? fd.y : k == 2 ? fd.z : fd.w;
                if (didx != DIDX_DEAD) {
                    double* y = (double*)(c.Yl + ((size_t)didx << 8));
                    double v = 0.0;
                    if ((h0.w >> k) & 1u) v = __ldcg(y);
                    v = fma(a.neg_kappa, close, v);
                    if (FUSED) *y = v; else __stcs(y, v);
                }
            }
        }
        if (flags & FLAG_READOUT) {          // terminal readout O_S (Eq. 15): one block per subset S
            // 2^(|S|-1): the continuation multiplicities of Lemma 7, applied once per output (exact)
            const double scale = (double)(1u << h0.y);
            if (valid) a.out[(size_t)h0.z * (size_t)a.batch + (size_t)b] = (a.neg_kappa * close) * scale;
        }
        mi = mi_n; bp = bp_n; pb ^= 1u;
    }
    cp_async_wait<0>();
}

__global__ void __launch_bounds__(MAX_WARPS * 32) cos_layer_kernel(const LayerArgs a)
{
    extern __shared__ __align__(128) double Gs[];
    __shared__ unsigned int s_next;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
    const uint32_t tile = blockIdx.x;

    const uint32_t gs_lane = (uint32_t)__cvta_generic_to_shared(Gs) + (uint32_t)lane * 8u;

    // Programmatic dependent launch: let the next layer's grid start (it only stages its table, which no layer
    // writes) while this grid drains; this grid in turn touches the slabs only after the previous one has completed.
    if (a.pdl) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // ---- stage the tile's propagator table Gs[slot][lane] with asynchronous copies (all in flight at once)
    const long long b = a.b0 + (long long)tile * TILE + lane;
    const bool valid = b < a.batch;
    if (threadIdx.x == 0) s_next = 0u;
    for (int s = warp; s < a.n_slots; s += W) {
        if (valid) cp_async8(gs_lane + (uint32_t)s * (TILE * 8u), a.G + (size_t)s * (size_t)a.batch + (size_t)b);
        else Gs[s * TILE + lane] = 0.0;
    }
    cp_async_commit();
    cp_async_wait<0>();
    __syncthreads();
    // continuation into the partner of the current endpoint (E2 with j = e) always comes with the counterterm one-cycle
    // E3 at the same destination: fold c3*sigma_lam into the diagonal of the staged table (Eq. 49 / 72, 77) and keep
    // the plain diagonal Gd for the cycle-closing factor (no shifts: Gd is a copy of the diagonal).
    for (int q = warp; q < a.nc * a.d; q += W) {
        const int lam = q / a.d, e = q - lam * a.d;
        const double sh = lam == 0 ? a.shift[0] : lam == 1 ? a.shift[1] : lam == 2 ? a.shift[2] : a.shift[3];
        const double g = Gs[((lam * a.d + e) * a.d + e) * TILE + lane];
        Gs[(a.n_slots + q) * TILE + lane] = g;
        if (a.has_shift) Gs[((lam * a.d + e) * a.d + e) * TILE + lane] = g + sh;
    }
    __syncthreads();

    if (a.pdl) asm volatile("griddepcontrol.wait;" ::: "memory");
    const uint32_t m_begin = blockIdx.y * a.masks_per_cta;
    const uint32_t m_end = min(a.n_masks, m_begin + a.masks_per_cta);
    const uint32_t rs_warp = (uint32_t)__cvta_generic_to_shared(Gs) + (uint32_t)(a.n_slots + a.nc * a.d) * (TILE * 8u) +
                             (uint32_t)warp * RECORD_SLOT_BYTES;
    layer_blocks<false>(a, m_begin, m_end, tile, s_next, gs_lane, rs_warp, lane, valid, b);
}

// ------------------------------------------------------------------------------------------------------
// Fused small-DAG kernel: ONE launch walks every layer.  A batch tile's states are touched by one CTA only, so the
// layers of a tile need nothing stronger than __syncthreads between them: grid = batch tiles, the CTA stages the table
// once, writes the layer-0 states (Eq. 66) itself and ping-pongs between two slabs of S_max states per tile (L2-resident;
// source rows are read with ld.global.cg so that no stale L1 line of the slab written two layers earlier is seen).
// Used when every layer is small (launch latency, not bandwidth, decides: orders n <= 6).
__global__ void __launch_bounds__(MAX_WARPS * 32) cos_fused_kernel(const FusedArgs f)
{
    extern __shared__ __align__(128) double Gs[];
    __shared__ unsigned int s_next;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
    const uint32_t tile = blockIdx.x;
    const uint32_t gs_lane = (uint32_t)__cvta_generic_to_shared(Gs) + (uint32_t)lane * 8u;
    const long long b = f.b0 + (long long)tile * TILE + lane;
    const bool valid = b < f.batch;
    if (threadIdx.x == 0) s_next = 0u;
    for (int s = warp; s < f.n_slots; s += W) {
        if (valid) cp_async8(gs_lane + (uint32_t)s * (TILE * 8u), f.G + (size_t)s * (size_t)f.batch + (size_t)b);
        else Gs[s * TILE + lane] = 0.0;
    }
    cp_async_commit();
    double* slab0 = f.ws + (size_t)tile * f.S_max * TILE;
    double* slab1 = f.ws + ((size_t)gridDim.x + tile) * f.S_max * TILE;
    for (uint32_t s = warp; s < f.layers[0].n_states; s += W) slab0[(size_t)s * TILE + lane] = 1.0;   // Eq. 66
    cp_async_wait<0>();
    __syncthreads();
    // keep the plain diagonal (cycle closing); the shifted one is rewritten per layer below
    for (int q = warp; q < f.nc * f.d; q += W) {
        const int lam = q / f.d, e = q - lam * f.d;
        Gs[(f.n_slots + q) * TILE + lane] = Gs[((lam * f.d + e) * f.d + e) * TILE + lane];
    }
    __syncthreads();
    const uint32_t rs_warp = (uint32_t)__cvta_generic_to_shared(Gs) + (uint32_t)(f.n_slots + f.nc * f.d) * (TILE * 8u) +
                             (uint32_t)warp * RECORD_SLOT_BYTES;
    LayerArgs a;
    a.G = f.G; a.batch = f.batch; a.b0 = f.b0; a.out = f.out; a.d = f.d; a.nc = f.nc; a.n_slots = f.n_slots;
    a.has_shift = f.has_shift;
    a.neg_kappa = f.neg_kappa; a.prefetch = 0; a.pdl = 0; a.S_src = f.S_max; a.S_dst = f.S_max; a.masks_per_cta = 0;
    for (int l = 0; l < f.n_layers; ++l) {
        if (f.has_shift && l <= 1) {         // c3 = -2 at layer 0, -1 afterwards (Eq. 72, 77)
            for (int q = warp; q < f.nc * f.d; q += W) {
                const int lam = q / f.d, e = q - lam * f.d;
                const double sg = lam == 0 ? f.sigma[0] : lam == 1 ? f.sigma[1] : lam == 2 ? f.sigma[2] : f.sigma[3];
                Gs[((lam * f.d + e) * f.d + e) * TILE + lane] = Gs[(f.n_slots + q) * TILE + lane] + (l == 0 ? -2.0 : -1.0) * sg;
            }
            __syncthreads();
        }
        const FusedLayer fl = f.layers[l];
        a.words = fl.words; a.mask_off = fl.mask_off; a.n_masks = fl.n_masks;
        a.X = (l & 1) ? slab1 : slab0; a.Y = (l & 1) ? slab0 : slab1;
        // slabs are addressed per tile already: tile index 0 inside layer_blocks
        layer_blocks<true>(a, 0u, fl.n_masks, 0u, s_next, gs_lane, rs_warp, lane, valid, b);
        __threadfence_block();
        __syncthreads();
        if (threadIdx.x == 0) s_next = 0u;
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------------
size_t layer_smem_bytes(int n_slots, int nc, int d, int warps_per_cta)
{
    return (size_t)(n_slots + nc * d) * TILE * sizeof(double) + (size_t)warps_per_cta * RECORD_SLOT_BYTES;
}

cudaError_t configure_layer_kernels()
{
    cudaError_t e = cudaFuncSetAttribute((const void*)cos_layer_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)LAYER_SMEM_MAX);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute((const void*)cos_fused_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)LAYER_SMEM_MAX);
}

// Launch shape: the CTA size that maximises resident warps per SM (ties: the smaller CTA).
cudaError_t pick_layer_shape(int nc, int d, int n_slots, int* warps_per_cta, int* ctas_per_sm)
{
    static const int cand[6] = {4, 6, 8, 10, 12, 16};
    int best_w = 0, best_total = 0, best_ctas = 0;
    for (int i = 0; i < 6; ++i) {
        if (cand[i] > MAX_WARPS) continue;
        const size_t smem = layer_smem_bytes(n_slots, nc, d, cand[i]);
        if (smem > LAYER_SMEM_MAX) continue;
        int nb = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, (const void*)cos_layer_kernel, cand[i] * 32, smem);
        if (e != cudaSuccess) return e;
        if (nb * cand[i] > best_total) { best_total = nb * cand[i]; best_w = cand[i]; best_ctas = nb; }
    }
    if (best_w == 0) return cudaErrorInvalidConfiguration;
    *warps_per_cta = best_w; *ctas_per_sm = best_ctas;
    return cudaSuccess;
}

cudaError_t layer_ctas_per_sm(int nc, int d, int n_slots, int warps_per_cta, int* ctas_per_sm)
{
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, (const void*)cos_layer_kernel, warps_per_cta * 32,
                                                         layer_smem_bytes(n_slots, nc, d, warps_per_cta));
}

cudaError_t launch_layer(const LayerArgs& a, uint32_t tiles, int warps_per_cta, cudaStream_t stream)
{
    if (a.n_masks == 0 || tiles == 0) return cudaSuccess;
    if (warps_per_cta < 1) warps_per_cta = 1;
    if (warps_per_cta > MAX_WARPS) warps_per_cta = MAX_WARPS;
    const uint32_t chunks = (a.n_masks + a.masks_per_cta - 1) / a.masks_per_cta;
    if (chunks > 65535u) return cudaErrorInvalidConfiguration;
    dim3 grid(tiles, chunks, 1), block(32 * warps_per_cta, 1, 1);
    const size_t smem = layer_smem_bytes(a.n_slots, a.nc, a.d, warps_per_cta);
    if (smem > LAYER_SMEM_MAX) return cudaErrorInvalidConfiguration;
    if (!a.pdl) {
        cos_layer_kernel<<<grid, block, smem, stream>>>(a);
        return cudaGetLastError();
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, cos_layer_kernel, a);
}

cudaError_t launch_fused(const FusedArgs& f, uint32_t tiles, int warps_per_cta, cudaStream_t stream)
{
    if (tiles == 0) return cudaSuccess;
    if (warps_per_cta > MAX_WARPS) warps_per_cta = MAX_WARPS;
    const size_t smem = layer_smem_bytes(f.n_slots, f.nc, f.d, warps_per_cta);
    if (smem > LAYER_SMEM_MAX) return cudaErrorInvalidConfiguration;
    cos_fused_kernel<<<tiles, 32 * warps_per_cta, smem, stream>>>(f);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------
__global__ void cos_fill_kernel(double* __restrict__ X, size_t n)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t step = (size_t)gridDim.x * blockDim.x;
    for (; i < n; i += step) X[i] = 1.0;
}

cudaError_t launch_fill_ones(double* X, size_t n, cudaStream_t stream)
{
    if (n == 0) return cudaSuccess;
    size_t blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    cos_fill_kernel<<<(unsigned)blocks, 256, 0, stream>>>(X, n);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------
// Propagator tabulation (north_star (2)).  One thread = (configuration, ordered vertex pair (i, j));
// it writes the n_blocks * n_sub^2 entries of that pair.  Arithmetic order is fixed with explicit
// round-to-nearest intrinsics (no FMA contraction) so that the result is reproducible bit for bit.
__global__ void cos_tabulate_kernel(const TabArgs a)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= a.batch) return;
    const int pair = blockIdx.y, i = pair / a.n, j = pair - i * a.n;
    const int xi = a.sites[((size_t)i * 2 + 0) * a.batch + c], yi = a.sites[((size_t)i * 2 + 1) * a.batch + c];
    const int xj = a.sites[((size_t)j * 2 + 0) * a.batch + c], yj = a.sites[((size_t)j * 2 + 1) * a.batch + c];
    int dx = (xi - xj) % a.L, dy = (yi - yj) % a.L;
    if (dx < 0) dx += a.L;
    if (dy < 0) dy += a.L;
    const int r = dx * a.L + dy;
    double dt = __dsub_rn(a.tau[(size_t)i * a.batch + c], a.tau[(size_t)j * a.batch + c]);
    double sign = 1.0;
    if (dt <= 0.0) { dt = __dadd_rn(dt, a.beta); sign = -1.0; }      // anti-periodic; equal times use 0^-
    const double step = a.beta / (double)(a.n_tau - 1);
    const double u = __ddiv_rn(dt, step);
    int k = (int)floor(u);
    if (k > a.n_tau - 2) k = a.n_tau - 2;
    const double w = __dsub_rn(u, (double)k);
    const int d = a.n * a.nsub, ns2 = a.nsub * a.nsub;
    for (int blk = 0; blk < a.n_blocks; ++blk)
        for (int s = 0; s < a.nsub; ++s)
            for (int s2 = 0; s2 < a.nsub; ++s2) {
                const double* t = a.T + (((size_t)blk * ns2 + (size_t)(s * a.nsub + s2)) * (size_t)(a.L * a.L) + r) * a.n_tau + k;
                const double g = __dadd_rn(__dmul_rn(__dsub_rn(1.0, w), __ldg(t)), __dmul_rn(w, __ldg(t + 1)));
                a.G[(((size_t)blk * d + (size_t)(i * a.nsub + s)) * d + (size_t)(j * a.nsub + s2)) * (size_t)a.batch + c] =
                    __dmul_rn(sign, g);
            }
}

cudaError_t launch_tabulate(const TabArgs& a, cudaStream_t stream)
{
    if (a.batch == 0) return cudaSuccess;
    dim3 block(128, 1, 1), grid((unsigned)((a.batch + 127) / 128), (unsigned)(a.n * a.n), 1);
    cos_tabulate_kernel<<<grid, block, 0, stream>>>(a);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------
// Many-configuration heat-bath weights (Eq. 6-7): one thread per configuration, subsets in increasing
// bitmask order, rounding order fixed (no contraction: products, one division and one addition per subset).
__global__ void cos_flux_kernel(const FluxArgs a)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= a.batch) return;
    const uint32_t n_sub = (1u << a.n) - 1u;
    double W = 0.0;
    for (uint32_t S = 1; S <= n_sub; ++S) {
        const int k = __popc(S);
        const size_t idx = (size_t)(S - 1u) * (size_t)a.batch + (size_t)c;
        if (!((a.order_mask >> k) & 1u)) {
            if (a.Phi) a.Phi[idx] = 0.0;
            continue;
        }
        double phi = __dmul_rn(a.lambda[k], __ldg(a.C + idx));
        if (a.Q) phi = __dmul_rn(phi, __ldg(a.Q + idx));
        if (a.Phi) a.Phi[idx] = phi;
        W = __dadd_rn(W, __ddiv_rn(fabs(phi), a.binom[k]));
    }
    a.W[c] = W;
}

cudaError_t launch_flux(const FluxArgs& a, cudaStream_t stream)
{
    if (a.batch == 0) return cudaSuccess;
    cos_flux_kernel<<<(unsigned)((a.batch + 127) / 128), 128, 0, stream>>>(a);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------
__global__ void cos_fp64_peak_kernel(double* sink, int iters, double a0, double b0)
{
    double acc[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = (double)(threadIdx.x + q);
    const double a = a0, bb = b0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 8; ++q) acc[q] = fma(acc[q], a, bb);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += acc[q];
    if (s == 123.456) sink[0] = s;          // never true; keeps the chain alive
}

cudaError_t measure_fp64_fma(double* fma_per_s)
{
    double* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, sizeof(double));
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0); cudaEventCreate(&t1);
    const int blocks = 148 * 8, threads = 256, iters = 1 << 16;
    cos_fp64_peak_kernel<<<blocks, threads>>>(sink, 1024, 0.999999, 1e-9);       // warm-up
    double best = 0.0;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(t0);
        cos_fp64_peak_kernel<<<blocks, threads>>>(sink, iters, 0.999999, 1e-9);
        cudaEventRecord(t1);
        e = cudaEventSynchronize(t1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        const double rate = (double)blocks * threads * 8.0 * (double)iters / (ms * 1e-3);
        if (rate > best) best = rate;
    }
    cudaEventDestroy(t0); cudaEventDestroy(t1);
    cudaFree(sink);
    if (e == cudaSuccess) e = cudaGetLastError();
    *fma_per_s = best;
    return e;
}

}  // namespace cosb
