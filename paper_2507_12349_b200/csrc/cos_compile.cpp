// cos_compile.cpp -- host-side DAG compiler (north_star subsystem (1)).
//
// Enumerates the reachable states of the reduced CoS / SB-CoS recurrence (forward sets F_l, Eq. 19-20),
// prunes them against the requested readouts (backward sets B_l, Eq. 21-24; K_l = F_l ^ B_l, Eq. 23),
// numbers them layer by layer (layer = total occupancy - 1) and emits the per-layer block/row program
// described in cos_compile.h.  Integer / structural work only; nothing numeric happens here.
//
// Transition rules (j ranges over labels >= r = min supp(m), Eq. 9-11):
//   E1  continue into an untouched interaction j, every sublattice s_j : multiplicity 2   (Eq. 11, Lemma 7)
//   E2  continue into the partner of a singly occupied interaction j   : multiplicity 1   (Eq. 11)
//   E3  counterterm one-cycle at the partner of the current endpoint   : -sigma_lambda    (Eq. 60, 72, 77)
//       (same destination as E2 with j = e; the kernel applies it as a diagonal correction)
//   E4  close (-kappa G[e][h]) and open the canonical head j = min{i: m_i = 1}, every colour (Eq. 12, 70-71)
//   readout when no interaction is singly occupied: out[S] += -kappa G[e][h] x               (Eq. 14-15)
#include "cos_compile.h"

#include <algorithm>
#include <cstring>
#include <map>
#include <utility>

namespace cosb {
namespace {

struct JEntry {
    uint8_t j_a;        // destination endpoint index (j, s_j)
    uint8_t mult2;      // 1: multiplicity 2 (untouched interaction), 0: multiplicity 1
    uint32_t dest_code; // mask code of the destination block
};

struct Builder {
    int n, nsub, d, nc;
    bool all_subsets, has_shift;
    std::vector<int32_t> index_of;              // mask code -> mask id (-1: not reached)
    std::vector<uint32_t> codes;                // mask id -> code (2 bits per interaction: 0, 1=(1,A), 2=(1,B), 3=full)
    std::vector<uint32_t> alive;                // [id*d + h_a] bitmask over e_a of live states (colour-independent)
    std::vector<uint32_t> row_base;             // [id*d + h_a] slab index of state (h_a, lambda=0, first e)
    std::vector<std::vector<uint32_t>> by_layer;

    static int cell(uint32_t code, int i) { return (code >> (2 * i)) & 3; }
    int root(uint32_t code) const { for (int i = 0; i < n; ++i) if (cell(code, i)) return i; return n; }
    int jmin(uint32_t code) const {             // canonical open interaction, Eq. 12
        for (int i = 0; i < n; ++i) { int c = cell(code, i); if (c == 1 || c == 2) return i; }
        return -1;
    }
    uint32_t full_set(uint32_t code) const {
        uint32_t S = 0;
        for (int i = 0; i < n; ++i) if (cell(code, i) == 3) S |= 1u << i;
        return S;
    }
    uint32_t get_mask(uint32_t code, int layer) {
        int32_t id = index_of[code];
        if (id >= 0) return (uint32_t)id;
        id = (int32_t)codes.size();
        index_of[code] = id;
        codes.push_back(code);
        alive.resize((size_t)(id + 1) * d, 0u);
        by_layer[layer].push_back((uint32_t)id);
        return (uint32_t)id;
    }
    int jlist(uint32_t code, JEntry* out) const {
        int k = 0;
        for (int i = root(code); i < n; ++i) {
            int c = cell(code, i);
            if (c == 0) {
                for (int s = 0; s < nsub; ++s) {
                    out[k].j_a = (uint8_t)(i * nsub + s); out[k].mult2 = 1;
                    out[k].dest_code = code | ((uint32_t)(1 + s) << (2 * i)); ++k;
                }
            } else if (c != 3) {
                out[k].j_a = (uint8_t)(i * nsub + (c - 1)); out[k].mult2 = 0;
                out[k].dest_code = code | (3u << (2 * i)); ++k;
            }
        }
        return k;
    }
    uint32_t state_index(uint32_t id, int h_a, int lam, int e_a) const {
        uint32_t a = alive[(size_t)id * d + h_a];
        uint32_t L = (uint32_t)__builtin_popcount(a);
        return row_base[(size_t)id * d + h_a] + (uint32_t)lam * L + (uint32_t)__builtin_popcount(a & ((1u << e_a) - 1u));
    }
};

}  // namespace

std::string compile_dag(int n, int nf, int nsub, const double* sigma, bool uniform_shift, bool all_subsets,
                        uint32_t order_mask, CompiledDag& out, EquivalenceStats* eq)
{
    const bool uniform = (sigma == nullptr) || uniform_shift;
    if (n < 1 || n > 12) return "n must be in [1, 12]";
    if (nsub != 1 && nsub != 2) return "n_sub must be 1 or 2";
    if (nf < 1) return "n_flavors must be >= 1";
    if (!uniform && nf > 4) return "unsupported: SB mode supports at most 4 flavours";
    if (n * nsub > 24) return "unsupported: n * n_sub must be <= 24";

    Builder b;
    b.n = n; b.nsub = nsub; b.d = n * nsub; b.nc = uniform ? 1 : nf;
    b.all_subsets = all_subsets; b.has_shift = (sigma != nullptr);
    const int d = b.d, nc = b.nc, NL = 2 * n;
    try {
        b.index_of.assign((size_t)1 << (2 * n), -1);
        b.by_layer.assign(NL, {});

        // ---- initial states (Eq. 66; reading G8 for the rooted branches): (r, s) head = endpoint, m = (1,s) e_r
        // requested subsets (Eq. 24): all-subset mode keeps S with |S| in the allowed orders U (order_mask bit |S|;
        // 0 = every order); a subset of order k has root r = min S <= n - k, so larger roots are never started
        if (all_subsets && order_mask == 0) order_mask = ((2u << n) - 1u) & ~1u;
        int k_min = n;
        if (all_subsets) { k_min = 1; while (k_min <= n && !((order_mask >> k_min) & 1u)) ++k_min; }
        if (all_subsets && k_min > n) return "order_mask selects no order in [1, n]";
        auto requested = [&](uint32_t S) {
            return all_subsets ? (bool)((order_mask >> __builtin_popcount(S)) & 1u) : S == ((1u << n) - 1u);
        };
        for (int r = 0; r < (all_subsets ? n - k_min + 1 : 1); ++r)
            for (int s = 0; s < nsub; ++s) {
                uint32_t id = b.get_mask((uint32_t)(1 + s) << (2 * r), 0);
                int a = r * nsub + s;
                b.alive[(size_t)id * d + a] |= 1u << a;
            }

        // ---- forward reachability, Eq. 19-20
        JEntry J[24];
        for (int l = 0; l + 1 < NL; ++l) {
            for (size_t k = 0; k < b.by_layer[l].size(); ++k) {
                const uint32_t id = b.by_layer[l][k], code = b.codes[id];
                const int nJ = b.jlist(code, J);
                uint32_t dest[24];
                for (int q = 0; q < nJ; ++q) dest[q] = b.get_mask(J[q].dest_code, l + 1);
                for (int h = 0; h < d; ++h) {
                    if (!b.alive[(size_t)id * d + h]) continue;
                    for (int q = 0; q < nJ; ++q) b.alive[(size_t)dest[q] * d + h] |= 1u << J[q].j_a;
                }
                const int jm = b.jmin(code);
                if (jm >= 0) {
                    bool any = false;
                    for (int h = 0; h < d; ++h) any = any || b.alive[(size_t)id * d + h];
                    if (any) {
                        const int fa = jm * nsub + (Builder::cell(code, jm) - 1);
                        uint32_t did = b.get_mask(code | (3u << (2 * jm)), l + 1);
                        b.alive[(size_t)did * d + fa] |= 1u << fa;
                    }
                }
            }
        }
        uint64_t unpruned = 0;
        for (uint32_t a : b.alive) unpruned += (uint64_t)__builtin_popcount(a) * nc;

        // ---- backward productivity, Eq. 21-24, then K_l = F_l ^ B_l (Eq. 23)
        const uint32_t FULL = (n == 16) ? 0xFFFFu : ((1u << n) - 1u);
        std::vector<uint32_t> prod(b.alive.size(), 0u);
        for (int l = NL - 1; l >= 0; --l) {
            for (uint32_t id : b.by_layer[l]) {
                const uint32_t code = b.codes[id];
                const int jm = b.jmin(code);
                const bool readout = (jm < 0) && requested(b.full_set(code));
                bool fresh_ok = false;
                if (jm >= 0 && l + 1 < NL) {
                    const int fa = jm * nsub + (Builder::cell(code, jm) - 1);
                    int32_t did = b.index_of[code | (3u << (2 * jm))];
                    fresh_ok = did >= 0 && ((prod[(size_t)did * d + fa] >> fa) & 1u);
                }
                const int nJ = (l + 1 < NL) ? b.jlist(code, J) : 0;
                for (int h = 0; h < d; ++h) {
                    const uint32_t a = b.alive[(size_t)id * d + h];
                    if (!a) continue;
                    bool p = readout || fresh_ok;
                    for (int q = 0; q < nJ && !p; ++q) {
                        int32_t did = b.index_of[J[q].dest_code];
                        p = did >= 0 && ((prod[(size_t)did * d + h] >> J[q].j_a) & 1u);
                    }
                    prod[(size_t)id * d + h] = p ? a : 0u;
                }
            }
        }
        b.alive.swap(prod);
        prod.clear(); prod.shrink_to_fit();

        // ---- numbering: layer slab order = [block (by mask code)][head][colour][endpoint]
        out = CompiledDag();
        out.n = n; out.nf = nf; out.nsub = nsub; out.d = d; out.nc = nc;
        out.n_blocks = uniform ? 1 : nf;
        out.uniform = uniform; out.all_subsets = all_subsets; out.order_mask = all_subsets ? order_mask : 0u; out.has_shift = (sigma != nullptr);
        out.kappa = uniform ? (double)nf : 1.0;
        out.n_out = all_subsets ? (int)FULL : 1;
        for (int l = 0; l < nc && sigma; ++l) out.sigma[l] = sigma[l];
        out.n_states_unpruned = unpruned;
        out.layers.assign(NL, LayerProgram());
        b.row_base.assign(b.alive.size(), 0u);
        for (int l = 0; l < NL; ++l) {
            auto& ids = b.by_layer[l];
            std::vector<uint32_t> keep;
            for (uint32_t id : ids) {
                bool any = false;
                for (int h = 0; h < d; ++h) any = any || b.alive[(size_t)id * d + h];
                if (any) keep.push_back(id);
            }
            std::sort(keep.begin(), keep.end(), [&](uint32_t x, uint32_t y) { return b.codes[x] < b.codes[y]; });
            ids.swap(keep);
            uint64_t counter = 0;
            for (uint32_t id : ids)
                for (int h = 0; h < d; ++h) {
                    const uint32_t a = b.alive[(size_t)id * d + h];
                    if (!a) continue;
                    b.row_base[(size_t)id * d + h] = (uint32_t)counter;
                    counter += (uint64_t)__builtin_popcount(a) * nc;
                }
            if (counter >= DIDX_DEAD) return "unsupported: a layer has more than 2^24 - 1 states (24-bit destination index)";
            out.layers[l].n_states = (uint32_t)counter;
            out.layers[l].n_masks = (uint32_t)ids.size();
        }

        // ---- optional analysis: future / past equivalence classes of the pruned DAG (Eq. 25-28)
        if (eq) {
            *eq = EquivalenceStats();
            // global numbering: layer offsets + index inside the layer; edges enumerated exactly as the emission does
            std::vector<uint64_t> layer_off(NL + 1, 0);
            for (int l = 0; l < NL; ++l) layer_off[l + 1] = layer_off[l] + out.layers[l].n_states;
            const uint64_t S = layer_off[NL];
            if (S > 60000000ull) return "unsupported: equivalence analysis is limited to 6e7 states";
            // an edge = (label, coefficient, other end): label = the factor SYMBOL (G_lambda[a][b], or the counterterm of
            // colour lambda); two edges carry the same operator iff label and integer coefficient agree (Eq. 17)
            struct Edge { uint32_t src, dst; uint32_t label; int32_t coeff; };
            std::vector<Edge> edges;
            std::vector<std::pair<uint32_t, uint64_t>> readouts;     // (state, label | out_idx << 32)
            const uint32_t SHIFT_LABEL = (uint32_t)(nc * d * d);
            for (int l = 0; l < NL; ++l)
                for (uint32_t id : b.by_layer[l]) {
                    const uint32_t code = b.codes[id];
                    const int jm = b.jmin(code);
                    const int nJ = (l + 1 < NL) ? b.jlist(code, J) : 0;
                    int32_t fresh_did = -1; uint32_t fresh_a = 0; bool fresh = false;
                    if (jm >= 0 && l + 1 < NL) {
                        fresh_a = (uint32_t)(jm * nsub + (Builder::cell(code, jm) - 1));
                        fresh_did = b.index_of[code | (3u << (2 * jm))];
                        fresh = fresh_did >= 0 && ((b.alive[(size_t)fresh_did * d + fresh_a] >> fresh_a) & 1u);
                    }
                    const bool readout = jm < 0 && requested(b.full_set(code));
                    for (int h = 0; h < d; ++h) {
                        const uint32_t a = b.alive[(size_t)id * d + h];
                        for (int e = 0; e < d && a; ++e) {
                            if (!((a >> e) & 1u)) continue;
                            for (int lam = 0; lam < nc; ++lam) {
                                const uint32_t src = (uint32_t)(layer_off[l] + b.state_index(id, h, lam, e));
                                for (int q = 0; q < nJ; ++q) {
                                    const int32_t did = b.index_of[J[q].dest_code];
                                    if (did < 0 || !((b.alive[(size_t)did * d + h] >> J[q].j_a) & 1u)) continue;
                                    const uint32_t dst = (uint32_t)(layer_off[l + 1] + b.state_index((uint32_t)did, h, lam, J[q].j_a));
                                    edges.push_back({src, dst, (uint32_t)((lam * d + e) * d + J[q].j_a), J[q].mult2 ? 2 : 1});
                                    if (b.has_shift && !J[q].mult2 && J[q].j_a == e)      // E3 shares E2's destination
                                        edges.push_back({src, dst, SHIFT_LABEL + (uint32_t)lam, l == 0 ? -2 : -1});
                                }
                                if (fresh)
                                    for (int l2 = 0; l2 < nc; ++l2)
                                        edges.push_back({src, (uint32_t)(layer_off[l + 1] + b.state_index((uint32_t)fresh_did, (int)fresh_a, l2, (int)fresh_a)),
                                                         (uint32_t)((lam * d + e) * d + h), -(int32_t)out.kappa});
                                if (readout)
                                    readouts.push_back({src, (uint64_t)((lam * d + e) * d + h) |
                                                                 ((uint64_t)(all_subsets ? b.full_set(code) : 1u) << 32)});
                            }
                        }
                    }
                }
            eq->n_states = S; eq->n_edges = edges.size() + readouts.size();
            // operator symbol = (label, integer coefficient) pair, interned into a dense id (< 2^31: bit 63 marks readouts);
            // the coefficient is a full int32 (-kappa = -N_f has no upper bound in uniform mode)
            std::map<std::pair<uint32_t, int32_t>, uint32_t> symbols;
            auto key = [&symbols](uint32_t label, int32_t coeff, uint32_t cls) {
                const auto it = symbols.emplace(std::make_pair(label, coeff), (uint32_t)symbols.size()).first;
                return ((uint64_t)it->second << 32) | (uint64_t)cls;
            };
            // future classes (Eq. 25-26): last layer first; signature = sorted (label, coefficient, class of the child)
            std::vector<std::vector<uint64_t>> sig(S);
            std::vector<uint32_t> cls(S, 0);
            for (auto& r : readouts) sig[r.first].push_back((1ull << 63) | r.second);
            std::vector<uint32_t> order(edges.size());
            for (size_t i = 0; i < edges.size(); ++i) order[i] = (uint32_t)i;
            std::stable_sort(order.begin(), order.end(), [&](uint32_t x, uint32_t y) { return edges[x].src > edges[y].src; });
            {
                size_t pos = 0;
                uint64_t n_cls = 0, n_edges_after = 0;
                for (int l = NL - 1; l >= 0; --l) {
                    // edges are sorted by decreasing source: the sources of layer l come after those of layer l + 1
                    while (pos < order.size() && edges[order[pos]].src >= layer_off[l]) {
                        const Edge& E = edges[order[pos++]];
                        sig[E.src].push_back(key(E.label, E.coeff, cls[E.dst]));
                    }
                    std::map<std::vector<uint64_t>, uint32_t> ids;
                    for (uint64_t x = layer_off[l]; x < layer_off[l + 1]; ++x) {
                        std::sort(sig[x].begin(), sig[x].end());
                        auto it = ids.find(sig[x]);
                        if (it == ids.end()) { it = ids.emplace(sig[x], (uint32_t)ids.size()).first; n_edges_after += sig[x].size(); }
                        cls[x] = (uint32_t)(layer_off[l] + it->second);
                        std::vector<uint64_t>().swap(sig[x]);
                    }
                    n_cls += ids.size();
                }
                eq->future_classes = n_cls; eq->edges_after_future_merge = n_edges_after;
            }
            // past classes (Eq. 27-28): first layer first; signature = sorted (label, coefficient, class of the parent);
            // the initial states (value 1, Eq. 66) share the empty signature
            std::stable_sort(order.begin(), order.end(), [&](uint32_t x, uint32_t y) { return edges[x].dst < edges[y].dst; });
            {
                size_t pos = 0;
                uint64_t n_cls = 0, n_edges_after = readouts.size();
                for (int l = 0; l < NL; ++l) {
                    while (pos < order.size() && edges[order[pos]].dst < layer_off[l + 1]) {
                        const Edge& E = edges[order[pos++]];
                        sig[E.dst].push_back(key(E.label, E.coeff, cls[E.src]));
                    }
                    std::map<std::vector<uint64_t>, uint32_t> ids;
                    for (uint64_t x = layer_off[l]; x < layer_off[l + 1]; ++x) {
                        std::sort(sig[x].begin(), sig[x].end());
                        auto it = ids.find(sig[x]);
                        if (it == ids.end()) { it = ids.emplace(sig[x], (uint32_t)ids.size()).first; n_edges_after += sig[x].size(); }
                        cls[x] = (uint32_t)(layer_off[l] + it->second);
                        std::vector<uint64_t>().swap(sig[x]);
                    }
                    n_cls += ids.size();
                }
                eq->past_classes = n_cls; eq->edges_after_past_merge = n_edges_after;
            }
        }

        // ---- emission
        const int HDR = out.hdr_words();
        for (int l = 0; l < NL; ++l) {
            LayerProgram& P = out.layers[l];
            P.mask_off.reserve(2 * (size_t)P.n_masks + 2);
            for (uint32_t id : b.by_layer[l]) {
                const uint32_t code = b.codes[id];
                const int jm = b.jmin(code);
                const int nJ = (l + 1 < NL) ? b.jlist(code, J) : 0;
                uint32_t flags = 0, fresh_a = 0, out_idx = 0;
                int32_t fresh_did = -1;
                if (jm >= 0 && l + 1 < NL) {
                    fresh_a = (uint32_t)(jm * nsub + (Builder::cell(code, jm) - 1));
                    fresh_did = b.index_of[code | (3u << (2 * jm))];
                    if (fresh_did >= 0 && ((b.alive[(size_t)fresh_did * d + fresh_a] >> fresh_a) & 1u)) flags |= FLAG_FRESH;
                }
                if (jm < 0 && requested(b.full_set(code))) {
                    flags |= FLAG_READOUT;
                    out_idx = all_subsets ? b.full_set(code) - 1u : 0u;
                }
                const bool need_close = flags != 0;
                uint32_t n_rows = 0, Lmax = 0;
                for (int h = 0; h < d; ++h) {
                    const uint32_t a = b.alive[(size_t)id * d + h];
                    if (a) { n_rows += nc; Lmax = std::max(Lmax, (uint32_t)__builtin_popcount(a)); }
                }
                const uint32_t e_words = (Lmax + 3) / 4, stride = 2 + e_words + (uint32_t)nJ;
                if (stride > 32) return "unsupported: row record exceeds 32 words";
                if (P.words.size() + HDR + (size_t)n_rows * stride >= 0xFFFFFFFFull) return "unsupported: layer program exceeds 2^32 words";
                P.mask_off.push_back((uint32_t)P.words.size());
                {   // first state of the block in the layer slab (block states are contiguous)
                    uint32_t first = P.n_states;
                    for (int h = 0; h < d; ++h)
                        if (b.alive[(size_t)id * d + h]) { first = b.row_base[(size_t)id * d + h]; break; }
                    P.mask_off.push_back(first);
                }
                P.words.push_back(n_rows | ((uint32_t)nJ << 16) | (flags << 24));
                // bits 24..: |S| - 1 of a readout block (the deferred multiplicity 2^(|S|-1), see cos_compile.h)
                const uint32_t sexp = (flags & FLAG_READOUT) ? (uint32_t)__builtin_popcount(b.full_set(code)) - 1u : 0u;
                P.words.push_back(stride | (e_words << 8) | (fresh_a << 16) | (sexp << 24));
                P.words.push_back(out_idx);
                for (int lam = 0; lam < nc; ++lam)
                    P.words.push_back((flags & FLAG_FRESH) ? b.state_index((uint32_t)fresh_did, (int)fresh_a, lam, (int)fresh_a)
                                                            : DIDX_DEAD);
                int32_t dest[24];
                for (int q = 0; q < nJ; ++q) dest[q] = b.index_of[J[q].dest_code];
                for (int h = 0; h < d; ++h) {
                    const uint32_t a = b.alive[(size_t)id * d + h];
                    if (!a) continue;
                    const uint32_t L = (uint32_t)__builtin_popcount(a);
                    for (int lam = 0; lam < nc; ++lam) {
                        P.words.push_back(b.row_base[(size_t)id * d + h] + (uint32_t)lam * L);
                        const uint32_t kh = ((a >> h) & 1u) ? (uint32_t)__builtin_popcount(a & ((1u << h) - 1u)) : 31u;
                        const size_t w_hdr = P.words.size();
                        P.words.push_back(0u);           // w1, filled below
                        uint32_t packed[6] = {0, 0, 0, 0, 0, 0};
                        int k = 0;
                        for (int e = 0; e < d; ++e)      // byte = lam*d + e_a: row index of G_lam[e_a][.] in the staged table
                            if ((a >> e) & 1u) { packed[k / 4] |= (uint32_t)(lam * d + e) << (8 * (k % 4)); ++k; }
                        for (uint32_t w = 0; w < e_words; ++w) P.words.push_back(packed[w]);
                        // live destinations only (pruned ones are dropped), the merged E2/E4 destination last
                        uint32_t n_live = 0, defer_word = 0, has_defer = 0;
                        for (int q = 0; q < nJ; ++q) {
                            const bool live = dest[q] >= 0 && ((b.alive[(size_t)dest[q] * d + h] >> J[q].j_a) & 1u);
                            if (!live) continue;
                            if (J[q].mult2) P.e1 += L; else P.e2 += L;
                            if ((flags & FLAG_FRESH) && (uint32_t)h == fresh_a && J[q].j_a == fresh_a) {
                                has_defer = 1; defer_word = (uint32_t)J[q].j_a << 24;
                                continue;
                            }
                            P.words.push_back(b.state_index((uint32_t)dest[q], h, lam, J[q].j_a) | ((uint32_t)J[q].j_a << 24));
                            ++n_live;
                        }
                        if (has_defer) P.words.push_back(defer_word);
                        for (uint32_t q = n_live + has_defer; q < (uint32_t)nJ; ++q) P.words.push_back(0u);
                        P.words[w_hdr] = L | ((uint32_t)h << 5) | ((uint32_t)lam << 10) | (kh << 12) | (n_live << 17) | (has_defer << 22);
                        const uint32_t alive_j = n_live + has_defer;
                        if (b.has_shift && l + 1 < NL)      // E3: states whose current interaction is singly occupied
                            for (int e = 0; e < d; ++e)
                                if (((a >> e) & 1u)) { int c = Builder::cell(code, e / nsub); if (c == 1 || c == 2) P.e3 += 1; }
                        if (flags & FLAG_FRESH) P.e4 += (uint64_t)L * nc;
                        if (flags & FLAG_READOUT) P.readout_edges += L;
                        P.n_fma += (uint64_t)L * (alive_j + (need_close ? 1u : 0u));
                    }
                }
                P.n_rows += n_rows;
                P.max_L = std::max(P.max_L, Lmax);
            }
            P.mask_off.push_back((uint32_t)P.words.size());
            P.mask_off.push_back(P.n_states);
            P.words.resize(P.words.size() + 64, 0u);          // padding: the kernel reads whole 32-word windows
            out.n_states += P.n_states; out.n_masks += P.n_masks; out.n_rows += P.n_rows;
            out.n_edges += P.e1 + P.e2 + P.e3 + P.e4; out.n_readout_edges += P.readout_edges; out.n_fma += P.n_fma;
            out.max_layer_states = std::max(out.max_layer_states, P.n_states);
            out.max_L = std::max(out.max_L, P.max_L);
        }
    } catch (const std::bad_alloc&) {
        return "out of host memory while compiling the DAG";
    }
    return "";
}

}  // namespace cosb
