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

// ---- program stream format (u32 words), one stream per layer ---------------------------------------
// block header (HDR_WORDS = 3 + nc words):
//   w0 : n_rows[0:16) | nJ[16:24) | flags[24:32)        flags: bit0 FRESH (close-and-open target alive),
//                                                               bit1 READOUT (terminal readout, Eq. 14-15)
//   w1 : row_stride[0:8) | e_words[8:16) | fresh_a[16:24) | (|S| - 1)[24:32) of a readout block
//   w2 : out_idx (readout row of out_dev)
//   w3..w3+nc-1 : destination state index (next layer) of the fresh-head state of colour lambda'
// row (row_stride = 2 + e_words + nJ words):
//   w0 : index of the row's first state in this layer's slab (row states are contiguous)
//   w1 : L[0:5) | h_a[5:10) | lambda[10:12) | k_h[12:17) | n_live[17:22) | defer[22]
//        k_h = position of the state with e_a == h_a in the row (31: none); its cycle-closing factor G[h][h] must
//        not carry the counterterm.  n_live = destinations that follow; defer = one more
//        destination word after them whose value merges with the fresh-head state (coalesced E2/E4 pair)
//   w2.. : lambda*d + e_a of the L states, one byte each (row of G_lambda[e_a][.] in the staged table)
//   then n_live (+ defer) words: dj = didx[0:24) | j_a[24:29)  (destination index in the next layer, destination
//        endpoint); pruned destinations (Eq. 23) are not listed; the row is padded to the block's common stride.
// The multiplicity 2 - m_j = 2 of a continuation into an untouched interaction (Lemma 7) is NOT applied per edge:
// every path into a state of mask m has taken exactly nz(m) - 1 such edges (nz = interactions with m_i >= 1; the root
// enters with factor 1), so the slabs hold x / 2^(nz(m)-1) and a readout of subset S is scaled by 2^(|S|-1), exactly.
static const uint32_t DIDX_MASK = 0x00FFFFFFu;
static const uint32_t DIDX_DEAD = 0x00FFFFFFu;     // fresh-head destination pruned (block header only)
static const uint32_t FLAG_FRESH = 1u, FLAG_READOUT = 2u;

struct LayerProgram {
    uint32_t n_states = 0, n_masks = 0, n_rows = 0, max_L = 0;
    std::vector<uint32_t> words;
    std::vector<uint32_t> mask_off;      // [n_masks + 1][2]: {word offset of the block header, first state of the block}
    uint64_t e1 = 0, e2 = 0, e3 = 0, e4 = 0, readout_edges = 0, n_fma = 0;
};

struct CompiledDag {
    int n = 0, nf = 0, nsub = 1, d = 0, nc = 1, n_blocks = 1, n_out = 1;
    bool uniform = true, all_subsets = false, has_shift = false;
    uint32_t order_mask = 0;             // all-subset mode: requested orders (bit k <=> |S| = k)
    double sigma[4] = {0, 0, 0, 0};
    double kappa = 1.0;
    std::vector<LayerProgram> layers;    // 2n layers; layer l holds the transitions l -> l+1 and the readouts at l
    uint64_t n_states = 0, n_states_unpruned = 0, n_masks = 0, n_rows = 0, n_edges = 0, n_readout_edges = 0, n_fma = 0;
    uint32_t max_layer_states = 0, max_L = 0;
    int hdr_words() const { return 3 + nc; }
};

// Future / past equivalence classes of the pruned DAG: states with the same future signature
// Sigma+ (Eq. 25-26: the set of (operator, class of the child) over their out-edges and readouts) can be merged by adding
// their values; states with the same past signature Sigma- (Eq. 27-28: (operator, class of the parent) over their
// in-edges) carry the same value and need to be stored once.  One backward and one forward refinement pass each.
struct EquivalenceStats {
    uint64_t n_states = 0, n_edges = 0;                           // E1..E4 uncoalesced + readout edges
    uint64_t future_classes = 0, edges_after_future_merge = 0;
    uint64_t past_classes = 0, edges_after_past_merge = 0;
};

// Returns "" on success, else an error message ("unsupported: ..." for a structural limit, otherwise out of memory).
// n in [1,12]; nsub in {1,2}.  sigma == nullptr -> uniform CoS without counterterm; sigma != nullptr -> SB-CoS with nf
// colours and shift-close weights sigma[0..nf), or, with uniform_shift, uniform CoS (one colour, loop factor nf) whose
// counterterm one-cycle has weight sigma[0] (reading G12).
// order_mask (all_subsets only): bit k set <=> subsets of order k are requested outputs (0 = every order).
// eq != nullptr: additionally fill the equivalence statistics (host time and memory ~ the edge count; <= 6e7 states).
std::string compile_dag(int n, int nf, int nsub, const double* sigma, bool uniform_shift, bool all_subsets,
                        uint32_t order_mask, CompiledDag& out, EquivalenceStats* eq = nullptr);

}  // namespace cosb
