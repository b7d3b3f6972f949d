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
    std::vector<uint32_t> colour_stride;        // [id] states of one colour of the block (slab order [block][colour][head][e])
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
        return row_base[(size_t)id * d + h_a] + (uint32_t)lam * colour_stride[id] +
               (uint32_t)__builtin_popcount(a & ((1u << e_a) - 1u));
    }
};

}  // namespace

std::string compile_dag(int n, int nf, int nsub, const double* sigma, bool uniform_shift, bool all_subsets,
                        uint32_t order_mask, CompiledDag& out)
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

        // ---- numbering: layer slab order = [block (by mask code)][colour][head][endpoint]
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
        b.colour_stride.assign(b.codes.size(), 0u);
        for (int l = 0; l < NL; ++l) {
            auto& ids = b.by_layer[l];
            std::vector<uint32_t> keep;
            for (uint32_t id : ids) {
                bool any = false;
                for (int h = 0; h < d; ++h) any = any || b.alive[(size_t)id * d + h];
                if (any) keep.push_back(id);
            }
            // Blocks of equal shape (live destination endpoints, heads) are neighbours in the slab and in the program: the
            // warps of an SM then run the same instance of the kernel's source loop at the same time (instruction cache).
            std::vector<uint32_t> shape(b.codes.size(), 0u);
            for (uint32_t id : keep) {
                const uint32_t code = b.codes[id];
                const int nJ = (l + 1 < NL) ? b.jlist(code, J) : 0;
                uint32_t n_heads = 0, n_cols = 0;
                for (int h = 0; h < d; ++h) n_heads += b.alive[(size_t)id * d + h] != 0u;
                for (int q = 0; q < nJ; ++q) {
                    const int32_t did = b.index_of[J[q].dest_code];
                    bool any = false;
                    for (int h = 0; h < d && !any && did >= 0; ++h)
                        any = b.alive[(size_t)id * d + h] && ((b.alive[(size_t)did * d + h] >> J[q].j_a) & 1u);
                    n_cols += any;
                }
                shape[id] = (n_cols << 8) | n_heads;
            }
            std::sort(keep.begin(), keep.end(), [&](uint32_t x, uint32_t y) {
                return shape[x] != shape[y] ? shape[x] < shape[y] : b.codes[x] < b.codes[y];
            });
            ids.swap(keep);
            uint64_t counter = 0;
            for (uint32_t id : ids) {
                uint32_t per_colour = 0;
                for (int h = 0; h < d; ++h) {
                    const uint32_t a = b.alive[(size_t)id * d + h];
                    if (!a) continue;
                    b.row_base[(size_t)id * d + h] = (uint32_t)counter + per_colour;
                    per_colour += (uint32_t)__builtin_popcount(a);
                }
                b.colour_stride[id] = per_colour;
                counter += (uint64_t)per_colour * nc;
            }
            if (counter >= DIDX_DEAD) return "unsupported: a layer has more than 2^32 - 2 states (32-bit destination index)";
            out.layers[l].n_states = (uint32_t)counter;
            out.layers[l].n_masks = (uint32_t)ids.size();
        }

        // ---- emission
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
                // heads of the block (colour-independent) and the destination columns that are live for at least one head
                int heads[24], n_heads = 0;
                uint32_t Lmax = 0;
                for (int h = 0; h < d; ++h) {
                    const uint32_t a = b.alive[(size_t)id * d + h];
                    if (a) { heads[n_heads++] = h; Lmax = std::max(Lmax, (uint32_t)__builtin_popcount(a)); }
                }
                int32_t dest[24];
                for (int q = 0; q < nJ; ++q) dest[q] = b.index_of[J[q].dest_code];
                auto live = [&](int h, int q) {
                    return dest[q] >= 0 && ((b.alive[(size_t)dest[q] * d + h] >> J[q].j_a) & 1u);
                };
                int cols[24], n_cols = 0;                       // live columns, increasing j_a (jlist is ordered by j_a)
                for (int q = 0; q < nJ; ++q) {
                    bool any = false;
                    for (int k = 0; k < n_heads && !any; ++k) any = live(heads[k], q);
                    if (any) cols[n_cols++] = q;
                }
                // column chunks of at most GROUP_MAX_COLS (balanced); a block without live columns still has one
                // (empty) chunk, which carries the cycle-closing sum
                const int n_chunks = std::max(1, (n_cols + GROUP_MAX_COLS - 1) / GROUP_MAX_COLS);
                P.mask_off.push_back((uint32_t)P.words.size());
                {   // first state of the block in the layer slab (block states are contiguous)
                    uint32_t first = P.n_states;
                    if (n_heads) first = b.row_base[(size_t)id * d + heads[0]];
                    P.mask_off.push_back(first);
                }
                const size_t w_block = P.words.size();
                P.words.push_back(flags << 24);                  // n_groups filled below
                // |S| - 1 of a readout block (the deferred multiplicity 2^(|S|-1), see cos_compile.h)
                P.words.push_back((flags & FLAG_READOUT) ? (uint32_t)__builtin_popcount(b.full_set(code)) - 1u : 0u);
                P.words.push_back(out_idx);
                P.words.push_back(0u);
                for (int lam = 0; lam < 4; ++lam)
                    P.words.push_back((lam < nc && (flags & FLAG_FRESH))
                                          ? b.state_index((uint32_t)fresh_did, (int)fresh_a, lam, (int)fresh_a) : DIDX_DEAD);
                uint32_t n_groups = 0, merged = 0;
                std::vector<uint32_t> rec_at;                    // word offsets of the block's records, in program order
                for (int ch = 0; ch < n_chunks; ++ch) {
                    const int c0 = n_cols * ch / n_chunks, c1 = n_cols * (ch + 1) / n_chunks, TJ = c1 - c0;
                    const int th_max = TJ <= TILE_A_COLS ? TILE_A_HEADS : TJ <= TILE_B_COLS ? TILE_B_HEADS : 1;
                    const int n_hgroups = (n_heads + th_max - 1) / th_max;
                    for (int lam = 0; lam < nc; ++lam)
                        for (int g = 0; g < n_hgroups; ++g) {
                            const int h0 = n_heads * g / n_hgroups, h1 = n_heads * (g + 1) / n_hgroups, TH = h1 - h0;
                            uint32_t emask = 0, jmask = 0;
                            for (int k = h0; k < h1; ++k) emask |= b.alive[(size_t)id * d + heads[k]];
                            for (int c = c0; c < c1; ++c) jmask |= 1u << J[cols[c]].j_a;
                            const uint32_t row_words = ((uint32_t)TJ + 1u) & ~1u;      // destination rows are 8-byte aligned
                            const uint32_t len = 4u + 4u * (uint32_t)TH + (((uint32_t)TH * row_words + 3u) & ~3u);
                            if (P.words.size() + len >= 0xFFFFFFF0ull) return "unsupported: layer program exceeds 2^32 words";
                            uint32_t n_src = 0;                                  // source states of the record
                            for (int k = h0; k < h1; ++k) n_src += (uint32_t)__builtin_popcount(b.alive[(size_t)id * d + heads[k]]);
                            rec_at.push_back((uint32_t)P.words.size());
                            P.words.push_back((uint32_t)TH | ((uint32_t)TJ << 3) | ((uint32_t)lam << 8) |
                                              ((need_close && ch == 0) ? 1u << 10 : 0u) | (n_src << 11) | ((len / 4u) << 24));
                            P.words.push_back(emask);
                            P.words.push_back(jmask);
                            P.words.push_back(b.row_base[(size_t)id * d + heads[h0]] + (uint32_t)lam * b.colour_stride[id]);
                            for (int k = h0; k < h1; ++k) {
                                const int h = heads[k];
                                P.words.push_back(b.row_base[(size_t)id * d + h] + (uint32_t)lam * b.colour_stride[id]);
                                P.words.push_back(b.alive[(size_t)id * d + h]);
                                P.words.push_back((uint32_t)h);
                                P.words.push_back(0u);
                            }
                            const uint32_t U = (uint32_t)__builtin_popcount(emask);
                            for (int k = h0; k < h1; ++k) {
                                const int h = heads[k];
                                const uint32_t L = (uint32_t)__builtin_popcount(b.alive[(size_t)id * d + h]);
                                for (int c = c0; c < c1; ++c) {
                                    const int q = cols[c];
                                    uint32_t w = DIDX_DEAD;
                                    if (live(h, q)) {
                                        if (J[q].mult2) P.e1 += L; else P.e2 += L;
                                        P.n_factor_loads_unshared += L;
                                        // the continuation into the canonical open interaction from its own head lands on the
                                        // fresh-head state (coalesced E2/E4 pair)
                                        // (same destination state as the block's fresh-head state of this colour; the
                                        // kernel adds the closing sum to it at the end of the block, header w3 bit lam)
                                        if ((flags & FLAG_FRESH) && (uint32_t)h == fresh_a && J[q].j_a == fresh_a) merged |= 1u << lam;
                                        w = b.state_index((uint32_t)dest[q], h, lam, J[q].j_a);
                                    }
                                    P.words.push_back(w);
                                }
                                if (TJ & 1) P.words.push_back(DIDX_DEAD);
                            }
                            while (P.words.size() & 3u) P.words.push_back(DIDX_DEAD);
                            P.n_fma += (uint64_t)TH * U * (uint64_t)TJ;
                            P.n_factor_loads += (uint64_t)U * (uint64_t)TJ;
                            ++n_groups;
                        }
                }
                // per-row bookkeeping that does not depend on the grouping
                for (int k = 0; k < n_heads; ++k) {
                    const uint32_t a = b.alive[(size_t)id * d + heads[k]];
                    const uint32_t L = (uint32_t)__builtin_popcount(a);
                    for (int lam = 0; lam < nc; ++lam) {
                        if (b.has_shift && l + 1 < NL)      // E3: states whose current interaction is singly occupied
                            for (int e = 0; e < d; ++e)
                                if (((a >> e) & 1u)) { int c = Builder::cell(code, e / nsub); if (c == 1 || c == 2) P.e3 += 1; }
                        if (flags & FLAG_FRESH) P.e4 += (uint64_t)L * nc;
                        if (flags & FLAG_READOUT) P.readout_edges += L;
                        if (need_close) { P.n_fma += L; P.n_factor_loads += L; P.n_factor_loads_unshared += L; }
                    }
                }
                // L2 look-ahead hints: record i names the source range of record i + GROUP_LOOKAHEAD of the same block
                for (size_t i = 0; i + GROUP_LOOKAHEAD < rec_at.size(); ++i) {
                    const uint32_t tgt = rec_at[i + GROUP_LOOKAHEAD];
                    const uint32_t cnt = (P.words[tgt] >> 11) & 0x7Fu;
                    P.words[rec_at[i]] |= ((cnt + 1u) / 2u) << 18;
                    P.words[rec_at[i] + 7] = P.words[tgt + 3];
                }
                if (n_groups > 0xFFFFu) return "unsupported: more than 65535 group records in one block";
                P.words[w_block] |= n_groups;
                P.words[w_block + 3] = merged;
                P.n_groups += n_groups;
                P.n_rows += (uint32_t)n_heads * nc;
                P.max_L = std::max(P.max_L, Lmax);
            }
            P.mask_off.push_back((uint32_t)P.words.size());
            P.mask_off.push_back(P.n_states);
            P.words.resize(P.words.size() + 64, 0u);          // padding: the kernel may touch the line after the last record
            out.n_states += P.n_states; out.n_masks += P.n_masks; out.n_rows += P.n_rows; out.n_groups += P.n_groups;
            out.n_edges += P.e1 + P.e2 + P.e3 + P.e4; out.n_readout_edges += P.readout_edges; out.n_fma += P.n_fma;
            out.n_factor_loads += P.n_factor_loads; out.n_factor_loads_unshared += P.n_factor_loads_unshared;
            out.max_layer_states = std::max(out.max_layer_states, P.n_states);
            out.max_L = std::max(out.max_L, P.max_L);
        }
    } catch (const std::bad_alloc&) {
        return "out of host memory while compiling the DAG";
    }
    return "";
}

}  // namespace cosb
