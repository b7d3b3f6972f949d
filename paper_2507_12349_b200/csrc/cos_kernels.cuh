// cos_kernels.cuh -- launch interface between the C-ABI (cos_capi.cu) and the kernels (cos_kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace cosb {

static const int TILE = 32;              // configurations per batch tile = one warp, lane = configuration
static const size_t LAYER_SMEM_MAX = 227 * 1024 - 1024;   // minus the static counter and the 128-byte alignment of the table

struct LayerArgs {
    const uint32_t* words;               // layer program (cos_compile.h)
    const uint32_t* mask_off;            // [n_masks+1][2]: {header word offset, first state}
    uint32_t n_masks, masks_per_cta;
    uint32_t n_words, n_out;             // extent of `words` (padding included) and of the output rows (self-check build)
    const double* X;                     // source slab  [tile][S_src][32]
    double* Y;                           // destination slab [tile][S_dst][32]
    uint32_t S_src, S_dst;
    const double* G;                     // caller's propagators [n_slots][batch]
    long long batch, b0;                 // total batch (row stride of G / out) and first configuration of this chunk
    double* out;                         // caller's output [n_out][batch]
    int d, n_slots;                      // n_slots = n_blocks * d * d
    double neg_kappa;                    // -kappa: -N_f (uniform) or -1 (SB)
    int prefetch;                        // > 0: per row, prefetch into L2 the source states this many states ahead; 0: off
    int pdl;                             // 1: launched with programmatic stream serialization (layers > 0)
    double shift[4];                     // c3 * sigma_lambda of THIS layer (c3 = -2 at layer 0, -1 after)
};

// Picks the instantiation (max row length, colours, shift) and launches one layer step.
// grid = (tiles, ceil(n_masks / masks_per_cta)); returns cudaGetLastError().
cudaError_t launch_layer(const LayerArgs& a, int max_L, int nc, bool shift, uint32_t tiles, int warps_per_cta,
                         cudaStream_t stream);
// Opt-in to > 48 KB dynamic shared memory for every instantiation, per-layer and fused (once per process).
cudaError_t configure_layer_kernels();
// staged table (+ plain diagonal in shift mode) of one batch tile
size_t layer_smem_bytes(int n_slots, int nc, int d, bool shift);
// CTA size with the most resident warps per SM, and the resident CTAs per SM for a given CTA size
cudaError_t pick_layer_shape(int max_L, int nc, int d, int n_slots, bool shift, int* warps_per_cta, int* ctas_per_sm);
cudaError_t layer_ctas_per_sm(int max_L, int nc, int d, int n_slots, bool shift, int warps_per_cta, int* ctas_per_sm);

// ---- fused small-DAG path: every layer in one launch (cos_fused_kernel)
struct FusedLayer { const uint32_t* words; const uint32_t* mask_off; uint32_t n_masks, n_states, n_words; };
struct FusedArgs {
    const FusedLayer* layers;            // device array [n_layers]
    int n_layers;
    double* ws;                          // two slabs [2][tiles][S_max][32]
    uint32_t S_max;
    const double* G; long long batch, b0; double* out;
    int d, n_slots;
    uint32_t n_out;
    double neg_kappa;
    double sigma[4];
};
cudaError_t configure_fused_kernels();
cudaError_t launch_fused(const FusedArgs& f, int max_L, int nc, bool shift, uint32_t tiles, int warps_per_cta,
                         cudaStream_t stream);

cudaError_t launch_fill_ones(double* X, size_t n_doubles, cudaStream_t stream);

struct TabArgs {
    const double* T; int L, nsub, n_blocks, n_tau; double beta;
    int n; const int* sites; const double* tau; long long batch; double* G;
};
cudaError_t launch_tabulate(const TabArgs& a, cudaStream_t stream);

struct FluxArgs {
    int n; uint32_t order_mask; double lambda[13], binom[13];
    const double* C; const double* Q; double* W; double* Phi; long long batch;
};
cudaError_t launch_flux(const FluxArgs& a, cudaStream_t stream);

// ---- determinant-polynomial route (cos_det.cu; Eq. 34-38)
#define COS_DET_MAX_N 12
struct DetArgs {
    int n, n_blocks, three;              // three = 1: flavours 0, 1, 2; 0: flavours 0 and 2 (the middle one absent)
    int dd;                              // 1: double-double arithmetic (workspace elements are {hi, lo} pairs), 0: fp64
    int nsub;                            // 1 square; 2 honeycomb: the launcher walks all 2^n sublattice assignments
    uint32_t assign;                     // current assignment (bit i = sublattice of vertex i)
    int accumulate;                      // moment kernel adds to H instead of overwriting it
    int blk[3];                          // propagator block of each flavour (all 0 when the matrices are flavour-uniform)
    double sigma[3];                     // shift-close weights (sigma[1] unused with two flavours)
    uint32_t level_off[COS_DET_MAX_N + 1];   // subsets of size k are order[level_off[k] .. level_off[k-1])
    const double* G; long long batch;
    uint32_t* order;                     // [2^n] subsets by decreasing size
    void* minors;                        // [n_blocks][2^n][batch] elements of the working precision
    void* H;                             // [2^n][batch]
    void* C;                             // [2^n][batch] connected values in the working precision
    double* out;                         // caller's output [2^n-1][batch], fp64
};
cudaError_t launch_det_route(const DetArgs& a, cudaStream_t stream);

cudaError_t measure_fp64_fma(double* fma_per_s);
cudaError_t read_check_failures(long long* total, long long* by_kind);

}  // namespace cosb
