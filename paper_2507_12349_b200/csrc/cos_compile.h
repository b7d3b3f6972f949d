// cos_compile.h -- host-side DAG compiler of the CoS / SB-CoS recurrence (internal header).
//
// State of the reduced ("R-form") recurrence, Eq. 3-4, 8-12, 79-80:
//     X = (h, s_h, e, s_e, lambda, m),   m_i in {0, (1,s), 2}
// The compiler groups states by occupancy mask m ("block") and by (head, colour) ("row"); all
// continuation sources of a destination are one row (tail-vector form) and every
// destination state receives all of its contributions from ONE source block, which is what lets the
// kernel write each state exactly once without atomics.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace cosb {

// ---- program stream format (u32 words, every section 16-byte aligned so that the kernel reads it with warp-uniform
// 128-bit loads), one stream per layer ----------------------------------------------------------------------
// Slab order of a layer: [block = occupancy mask, by code][colour][head][endpoint].
// block header (HDR_WORDS = 8 words = two uint4):
//   w0 : n_groups[0:16) | flags[24:32)     flags: bit0 FRESH (close-and-open target alive),
//                                                  bit1 READOUT (terminal readout, Eq. 14-15)
//   w1 : (|S| - 1) of a readout block (the deferred multiplicity 2^(|S|-1), see below)
//   w2 : out_idx (readout row of out_dev)
//   w3 : bit lambda: a row of the block stores its continuation into the fresh-head state of colour lambda (the
//        coalesced E2/E4 pair: continuation from the canonical open interaction's own head); the kernel
//        then ADDS the closing sum to that state at the end of the block instead of overwriting it
//   w4..w7 : destination state index (next layer) of the fresh-head state of colour lambda' (DIDX_DEAD: pruned / unused)
// group record: up to GROUP_MAX_HEADS rows (heads) of ONE colour of the block that share the factor loads -- the
// factor-application sharing of PAPER.md Eq. 29-31: G_lambda[e][j] does not depend on the head, so one staged factor
// feeds the rows of all heads of the group (N_mult = min(|S_f|, |D_f|) -> one load per group instead of one per row):
//   q0 : g0 | emask | jmask | first
//        g0    = TH[0:3) | TJ[3:8) | lambda[8:10) | do_close[10] | n_src[11:18) | ahead2[18:24) | len4[24:32)
//                (n_src = source states of the record, len4 = record length in uint4 units; ahead2 * 2 states starting
//                at slab index `ahead` below are the sources of the record GROUP_LOOKAHEAD records later in this block:
//                the kernel prefetches them into L2 when it starts this record; 0 = nothing to prefetch)
//        emask = union over the heads of their live current endpoints e_a (bit e_a)
//        jmask = destination endpoints j_a of the TJ columns of this record (bit j_a), in increasing order
//        first = slab index of the group's first state (its states are contiguous: heads in increasing order)
//   TH x qh : base | alive | h_a | ahead   base = slab index of the head's first state, alive = its live endpoints (bit
//        e_a); ahead: look-ahead range start (first head only, see g0)
//   TH rows of TJ destination words, each row padded to an even number of words (and the record to a multiple of 4):
//        index of the destination state in the next layer's slab, or DIDX_DEAD (pruned, Eq. 23, or padding).
//   Register tiles of the kernel: up to TILE_A_HEADS heads when the block has at most TILE_A_COLS live destination
//   endpoints, up to TILE_B_HEADS heads for at most TILE_B_COLS, else one head x GROUP_MAX_COLS endpoints.  Blocks with more than GROUP_MAX_COLS live
//   destination endpoints are split into column chunks (one set of records per chunk; do_close is set in the first
//   chunk only, so that the cycle-closing sum is taken once).
// The multiplicity 2 - m_j = 2 of a continuation into an untouched interaction (Lemma 7) is NOT applied per edge:
// every path into a state of mask m has taken exactly nz(m) - 1 such edges (nz = interactions with m_i >= 1; the root
// enters with factor 1), so the slabs hold x / 2^(nz(m)-1) and a readout of subset S is scaled by 2^(|S|-1), exactly.
static const uint32_t DIDX_DEAD = 0xFFFFFFFFu;     // pruned destination
static const uint32_t FLAG_FRESH = 1u, FLAG_READOUT = 2u;
static const int HDR_WORDS = 8;
static const int TILE_A_HEADS = 4, TILE_A_COLS = 6;    // register tile A: 4 heads x 6 destination endpoints
static const int TILE_B_HEADS = 2, TILE_B_COLS = 8;    // register tile B: 2 heads x 8 endpoints; tile C: 1 head x GROUP_MAX_COLS
static const int GROUP_MAX_HEADS = 4;                  // rows sharing one factor load
static const int GROUP_MAX_COLS = 12;                  // destination columns of one record
static const int GROUP_LOOKAHEAD = 1;                  // L2 look-ahead distance in records

struct LayerProgram {
    uint32_t n_states = 0, n_masks = 0, n_rows = 0, n_groups = 0, max_L = 0;
    std::vector<uint32_t> words;
    std::vector<uint32_t> mask_off;      // [n_masks + 1][2]: {word offset of the block header, first state of the block}
    uint64_t e1 = 0, e2 = 0, e3 = 0, e4 = 0, readout_edges = 0, n_fma = 0;
    uint64_t n_factor_loads = 0, n_factor_loads_unshared = 0;   // staged-factor loads per configuration with / without Eq. 29-31
};

struct CompiledDag {
    int n = 0, nf = 0, nsub = 1, d = 0, nc = 1, n_blocks = 1, n_out = 1;
    bool uniform = true, all_subsets = false, has_shift = false;
    uint32_t order_mask = 0;             // all-subset mode: requested orders (bit k <=> |S| = k)
    double sigma[4] = {0, 0, 0, 0};
    double kappa = 1.0;
    std::vector<LayerProgram> layers;    // 2n layers; layer l holds the transitions l -> l+1 and the readouts at l
    uint64_t n_states = 0, n_states_unpruned = 0, n_masks = 0, n_rows = 0, n_groups = 0, n_edges = 0, n_readout_edges = 0, n_fma = 0;
    uint64_t n_factor_loads = 0, n_factor_loads_unshared = 0;
    uint32_t max_layer_states = 0, max_L = 0;
};

// Returns "" on success, else an error message ("unsupported: ..." for a structural limit, otherwise out of memory).
// n in [1,12]; nsub in {1,2}.  sigma == nullptr -> uniform CoS without counterterm; sigma != nullptr -> SB-CoS with nf
// colours and shift-close weights sigma[0..nf), or, with uniform_shift, uniform CoS (one colour, loop factor nf) whose
// counterterm one-cycle has weight sigma[0] (reading G12).
// order_mask (all_subsets only): bit k set <=> subsets of order k are requested outputs (0 = every order).
std::string compile_dag(int n, int nf, int nsub, const double* sigma, bool uniform_shift, bool all_subsets,
                        uint32_t order_mask, CompiledDag& out);

}  // namespace cosb
