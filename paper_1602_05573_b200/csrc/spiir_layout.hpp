// Host-side bank layout for the SPIIR filter kernels (north_star subsystem (1)
// "parameter array ... aligned and continuous ... coalesed memory access").
//
// A template's filters are sorted by delay, then dealt to "groups" of 32 (one filter per lane of a
// warp for one register slot f).  All 32 lanes of a group read their delayed input from shared memory in the same
// instruction, NC floats each, served in NC phases of 32/NC lanes; a phase is conflict-free iff the lanes' keys
// ceil(d / NC) mod (32 / NC) are distinct (or the delays equal).  The dealing first builds as many perfect phases as
// the key histogram allows and spreads the rest evenly, which keeps the average conflict degree near 1.4 / 1.2 / 1.1
// for NC = 1 / 2 / 4 and uniformly random delays (3.4 undealt, NC = 1).
// F consecutive groups form a warp tile (32 lanes x F register slots); tiles are padded with null
// filters (a1 = b0 = 0) whose delay copies a real filter of the same phase (same address = broadcast).
// Templates of <= 16 F filters can instead share a tile in aligned segments of 4, 8 or 16 lanes (pack_small).
//
// The layout of a template is a pure function of that template's own (a1, b0, d) arrays, so results are
// bitwise independent of the template's position in the bank (invariants).
#pragma once
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>

namespace spiir {

constexpr int kWarp = 32;

struct WarpWork {        // what one warp does in one round of one CTA item
    int32_t tile;        // warp tile index into the slot arrays, -1 = idle
    int32_t row;         // template index = SNR row
    int32_t first;       // first warp of this template in the round
    int32_t count;       // number of warps of this template in the round
};

struct HostLayout {
    int F = 0;                          // register slots (filters) per thread
    int W = 0;                          // warps of one CTA = warp tiles processed side by side
    int NC = 1;                         // shifted window copies = floats per shared-memory load
    int64_t n_tiles = 0;                // warp tiles
    int64_t n_slots = 0;                // n_tiles * F * 32
    std::vector<float> ar;              // [n_slots] Re a1
    std::vector<float> ai;              // [n_slots] Im a1 (the kernels build the (-Im, +Im) operand of the cross term)
    std::vector<float> b;               // [2*n_slots] (Re b0, Im b0)
    std::vector<int32_t> dly;           // [n_slots]
    // The device copy of the coefficients: one contiguous record per warp tile,
    //   [ar: F x 32][ai: F x 32][b: F x 32 (re, im) pairs][delay: F x 32 as int bits]  = 5 F x 32 floats,
    // so that a warp reaches everything it needs for a tile from one base address (5 F consecutive cache lines).
    std::vector<float> coef;
    std::vector<int64_t> slot_of_filter;  // [K] caller's filter index -> slot
    std::vector<int64_t> tile_begin;    // [T+1] first tile of each template
    // work list: items (one CTA at a time), each with >= 1 rounds of W warp entries
    std::vector<int32_t> item_round0;   // [n_items+1] first round of each item
    std::vector<WarpWork> work;         // [n_rounds * W]
    bool segmented = false;             // some warp tiles hold several small templates (tile_begin is then not a CSR)
    std::vector<int32_t> canon;         // [2W] (first, count) of every warp position when uniform_groups, else (-1, 0)
    bool uniform_groups = true;         // every warp position has the same (first, count) in all rounds it is active in
    double avg_conflict_degree = 0.0;   // mean over load phases of the max key multiplicity (diagnostic)
};

// Deal the delay-sorted filters `order` (indices into d) of one template into G groups of <= 32 lanes.
// A group is read with one shared-memory load instruction of NC floats per lane (NC = 1, 2, 4 =
// LDS.32/.64/.128 from NC shifted copies of the window); the hardware serves it in NC phases of
// P = 32/NC consecutive lanes, and a phase is conflict-free iff its lanes' aligned addresses fall into
// distinct NC-word bank groups, i.e. iff key(d) = ceil(d / NC) mod P is distinct (calls that start at a
// sample index that is a multiple of NC; other alignments stay correct and may conflict).
// Returns group-major list: out[g] = filter indices of group g, lanes in phase order.
inline int conflict_key(int32_t d, int NC, int P) { return (int)(((int64_t)d + NC - 1) / NC % P); }

inline void deal_groups(const int32_t* d, const std::vector<int64_t>& order, int G, int NC,
                        std::vector<std::vector<int64_t>>& out, double& degree_sum, int64_t& n_phases)
{
    const int P = kWarp / NC;              // lanes per phase = number of bank groups
    const int NP = G * NC;                 // phases to fill
    std::vector<std::vector<int64_t>> ph(NP);
    std::vector<std::vector<int64_t>> bucket(P);
    for (int64_t k : order) bucket[conflict_key(d[k], NC, P)].push_back(k);
    std::vector<size_t> head(P, 0);
    const int64_t K = (int64_t)order.size();
    // phase 1: perfect phases (one filter of every key), only full phases of P
    size_t perfect = bucket[0].size();
    for (int r = 1; r < P; ++r) perfect = std::min(perfect, bucket[r].size());
    perfect = std::min<size_t>(perfect, (size_t)(K / P));
    perfect = std::min<size_t>(perfect, (size_t)NP);
    for (size_t g = 0; g < perfect; ++g)
        for (int r = 0; r < P; ++r) ph[g].push_back(bucket[r][head[r]++]);
    // phase 2: spread the remainder evenly over the remaining phases: least multiplicity of the
    // key first, then emptiest phase, then lowest index; fullest keys first
    const int G2 = NP - (int)perfect;
    if (G2 > 0) {
        std::vector<int> rorder(P);
        std::iota(rorder.begin(), rorder.end(), 0);
        std::stable_sort(rorder.begin(), rorder.end(), [&](int a, int b) {
            return bucket[a].size() - head[a] > bucket[b].size() - head[b];
        });
        std::vector<int> fill(G2, 0);
        std::vector<int> mult((size_t)G2 * P, 0);
        // capacity per phase: all but the last phases are full, so that padding lands at the end
        const int64_t rem = K - (int64_t)perfect * P;
        std::vector<int> cap(G2, 0);
        {
            int64_t left = rem;
            for (int g = 0; g < G2; ++g) { cap[g] = (int)std::min<int64_t>(P, left); left -= cap[g]; }
        }
        for (int r : rorder) {
            while (head[r] < bucket[r].size()) {
                int best = -1;
                for (int g = 0; g < G2; ++g) {
                    if (fill[g] >= cap[g]) continue;
                    if (best < 0 || mult[(size_t)g * P + r] < mult[(size_t)best * P + r] ||
                        (mult[(size_t)g * P + r] == mult[(size_t)best * P + r] && fill[g] < fill[best]))
                        best = g;
                }
                ph[perfect + best].push_back(bucket[r][head[r]++]);
                ++fill[best];
                ++mult[(size_t)best * P + r];
            }
        }
    }
    // groups = NC consecutive phases; a short phase is followed only by empty ones
    out.assign(G, {});
    std::vector<int> cnt(P);
    for (int q = 0; q < NP; ++q) {
        if (ph[q].empty()) continue;
        std::fill(cnt.begin(), cnt.end(), 0);
        int mx = 0;
        for (int64_t k : ph[q]) mx = std::max(mx, ++cnt[conflict_key(d[k], NC, P)]);
        degree_sum += mx;
        ++n_phases;
        out[q / NC].insert(out[q / NC].end(), ph[q].begin(), ph[q].end());
    }
}

// A small template in a shared tile: its K_t filters go into `rows` register slots of w lanes each.  The w lanes of a row
// are read by the same load instruction (they sit inside one phase, or make up one, for w <= 32 / NC), so a row should hold
// distinct keys: fullest key classes first, every filter into the row that has the fewest of its key, then the emptiest,
// then the lowest; all rows but the last are full, so that the padding lands at the end.  Delay-sorted filters are dealt
// badly by position alone: K_t uniform delays over D samples are D / K_t apart, which is a multiple of the bank-group
// period as often as not.  The arrangement is a function of the template's own filters only (and of the bank-wide NC).
inline void deal_rows(const int32_t* d, const std::vector<int64_t>& order, int rows, int w, int NC,
                      std::vector<std::vector<int64_t>>& out)
{
    const int P = kWarp / NC;
    const int U = std::min(w, P);            // lanes dealt together: a whole phase, or the template's part of one
    const int per_row = w / U, units = rows * per_row;
    std::vector<std::vector<int64_t>> bucket(P), unit(units);
    for (int64_t k : order) bucket[conflict_key(d[k], NC, P)].push_back(k);
    std::vector<int> rorder(P);
    std::iota(rorder.begin(), rorder.end(), 0);
    std::stable_sort(rorder.begin(), rorder.end(), [&](int a, int b) { return bucket[a].size() > bucket[b].size(); });
    std::vector<int> cap(units, 0), fill(units, 0), mult((size_t)units * P, 0), deg(units, 0);
    {
        int64_t left = (int64_t)order.size();
        for (int g = 0; g < units; ++g) { cap[g] = (int)std::min<int64_t>(U, left); left -= cap[g]; }
    }
    // A whole phase costs as many wavefronts as its most frequent key (its degree): a filter that has to double up goes where
    // the degree does not grow (a phase that already holds a double), then where its key is rarest, then to the emptiest.
    // A template that fills only part of a phase (w < P) shares it with neighbours it does not know: there the doubles are
    // spread evenly instead (rarest key, then emptiest), which measures better than concentrating them.
    const bool whole = (w >= P);
    for (int r : rorder)
        for (int64_t k : bucket[r]) {
            int best = -1, best_grow = 0;
            for (int g = 0; g < units; ++g) {
                if (fill[g] >= cap[g]) continue;
                const int m = mult[(size_t)g * P + r];
                const int grow = whole ? std::max(deg[g], m + 1) - deg[g] : 0;
                if (best < 0 || grow < best_grow || (grow == best_grow && (m < mult[(size_t)best * P + r] ||
                    (m == mult[(size_t)best * P + r] && fill[g] < fill[best])))) {
                    best = g;
                    best_grow = grow;
                }
            }
            unit[best].push_back(k);
            ++fill[best];
            deg[best] = std::max(deg[best], ++mult[(size_t)best * P + r]);
        }
    // lanes of a unit in delay order (ties by caller index): any order is equally conflict-free; a row = per_row units
    out.assign(rows, {});
    for (int g = 0; g < units; ++g) {
        std::sort(unit[g].begin(), unit[g].end(), [&](int64_t x, int64_t y) { return d[x] != d[y] ? d[x] < d[y] : x < y; });
        out[g / per_row].insert(out[g / per_row].end(), unit[g].begin(), unit[g].end());
    }
}

// Lanes a small template occupies in a shared ("segmented") warp tile: the smallest of 4, 8, 16 whose lanes x F
// register slots hold its K_t filters; 32 = a template that gets warp tiles of its own (PAPER.md:L333-L335 maps
// templates of <= 32 filters to one warp; here several of them share one warp so that every lane still runs F filters).
inline int segment_lanes(int64_t Kt, int F, bool pack_small)
{
    if (!pack_small) return kWarp;
    for (int w : {4, 8, 16})
        if ((int64_t)w * F >= Kt) return w;
    return kWarp;
}

inline HostLayout build_layout(int32_t T, const int64_t* off, const float* a1, const float* b0,
                               const int32_t* d, int F, int W, int NC = 1, bool pack_small = false)
{
    HostLayout L;
    L.F = F;
    L.W = W;
    L.NC = NC;
    const int64_t K = off[T];
    L.tile_begin.resize((size_t)T + 1);
    int64_t tiles = 0;
    const int64_t per_tile = (int64_t)kWarp * F;
    // tile of every template; small templates of one size class that follow each other share a tile
    std::vector<int> seg_w((size_t)T, kWarp), seg_idx((size_t)T, 0);
    std::vector<int> tile_nseg;                       // templates in a tile (0 for regular tiles)
    {
        int open_w = 0, open_used = 0;
        int64_t open_tile = -1;
        for (int32_t t = 0; t < T; ++t) {
            const int64_t Kt = off[t + 1] - off[t];
            const int w = segment_lanes(Kt, F, pack_small);
            seg_w[t] = w;
            if (w == kWarp) {
                open_w = 0;
                L.tile_begin[t] = tiles;
                const int64_t nt = (Kt + per_tile - 1) / per_tile;
                tiles += nt;
                tile_nseg.resize((size_t)tiles, 0);
            } else {
                if (open_w != w || open_used == kWarp / w) {
                    open_tile = tiles++;
                    tile_nseg.resize((size_t)tiles, 0);
                    open_w = w;
                    open_used = 0;
                }
                L.tile_begin[t] = open_tile;
                seg_idx[t] = open_used++;
                tile_nseg[(size_t)open_tile] = open_used;
                L.segmented = true;
            }
        }
    }
    L.tile_begin[T] = tiles;
    L.n_tiles = tiles;
    L.n_slots = tiles * per_tile;
    L.ar.assign((size_t)L.n_slots, 0.f);
    L.ai.assign((size_t)L.n_slots, 0.f);
    L.b.assign((size_t)L.n_slots * 2, 0.f);
    L.dly.assign((size_t)L.n_slots, 0);
    L.slot_of_filter.assign((size_t)K, -1);

    double degree_sum = 0.0;
    int64_t n_phases = 0;
    std::vector<int64_t> order;
    std::vector<std::vector<int64_t>> groups;
    for (int32_t t = 0; t < T; ++t) {
        const int64_t k0 = off[t], Kt = off[t + 1] - off[t];
        order.resize((size_t)Kt);
        std::iota(order.begin(), order.end(), k0);
        std::stable_sort(order.begin(), order.end(), [&](int64_t x, int64_t y) { return d[x] < d[y]; });
        if (seg_w[t] < kWarp) {
            // small template: lanes [seg * w, seg * w + w) of a shared tile; its filters dealt to the F rows of those lanes
            const int w = seg_w[t];
            const int64_t tile = L.tile_begin[t];
            deal_rows(d, order, F, w, NC, groups);
            for (int g = 0; g < F; ++g)
                for (int l = 0; l < w; ++l) {
                    const int64_t s = (tile * F + g) * kWarp + (int64_t)seg_idx[t] * w + l;
                    if (l < (int)groups[g].size()) {
                        const int64_t k = groups[g][(size_t)l];
                        L.ar[s] = a1[2 * k];
                        L.ai[s] = a1[2 * k + 1];
                        L.b[2 * s] = b0[2 * k];
                        L.b[2 * s + 1] = b0[2 * k + 1];
                        L.dly[s] = d[k];
                        L.slot_of_filter[k] = s;
                    } else {
                        // null filter: the address of a real lane of the row (broadcast), else any valid window position
                        L.dly[s] = groups[g].empty() ? d[order[0]] : d[groups[g][0]];
                    }
                }
            continue;
        }
        const int64_t nt = (Kt + per_tile - 1) / per_tile;
        const int G = (int)(nt * F);
        deal_groups(d, order, G, NC, groups, degree_sum, n_phases);
        for (int g = 0; g < G; ++g) {
            if (groups[g].empty()) continue;
            // lanes in delay order inside the group (any order is equally conflict-free)
            const int64_t slot0 = (L.tile_begin[t] * F + g) * kWarp;
            for (size_t l = 0; l < groups[g].size(); ++l) {
                const int64_t k = groups[g][l], s = slot0 + (int64_t)l;
                L.ar[s] = a1[2 * k];
                L.ai[s] = a1[2 * k + 1];
                L.b[2 * s] = b0[2 * k];
                L.b[2 * s + 1] = b0[2 * k + 1];
                L.dly[s] = d[k];
                L.slot_of_filter[k] = s;
            }
            for (size_t l = groups[g].size(); l < (size_t)kWarp; ++l) {   // null filters: broadcast read
                const size_t first = l / (size_t)(kWarp / NC) * (size_t)(kWarp / NC);   // first lane of the phase
                L.dly[slot0 + (int64_t)l] = d[groups[g][first < groups[g].size() ? first : 0]];
            }
        }
        // entirely empty groups of the last tile: point them at the template's smallest delay
        for (int g = 0; g < G; ++g)
            if (groups[g].empty())
                for (int l = 0; l < kWarp; ++l) L.dly[(L.tile_begin[t] * F + g) * kWarp + l] = d[order[0]];
    }
    if (L.segmented) {
        // conflict statistics of the shared tiles (their lanes are not dealt: neighbours' delays are independent)
        std::vector<char> real((size_t)L.n_slots, 0);
        for (int64_t k = 0; k < K; ++k) real[(size_t)L.slot_of_filter[k]] = 1;
        const int P = kWarp / NC;
        std::vector<int> cnt(P);
        for (int64_t tile = 0; tile < tiles; ++tile) {
            if (!tile_nseg[(size_t)tile]) continue;
            for (int g = 0; g < F * NC; ++g) {
                const int64_t s0 = (tile * F + g / NC) * kWarp + (int64_t)(g % NC) * P;
                std::fill(cnt.begin(), cnt.end(), 0);
                int mx = 0;
                for (int l = 0; l < P; ++l)
                    if (real[(size_t)(s0 + l)]) mx = std::max(mx, ++cnt[conflict_key(L.dly[(size_t)(s0 + l)], NC, P)]);
                if (mx) { degree_sum += mx; ++n_phases; }
            }
        }
    }
    L.avg_conflict_degree = n_phases ? degree_sum / (double)n_phases : 0.0;

    // Work list.  Templates with <= W tiles share an item round with their neighbours (greedy, in bank
    // order); a template with more tiles gets an item of its own with several accumulate rounds.
    L.item_round0.push_back(0);
    std::vector<WarpWork> cur;
    auto flush = [&]() {
        if (cur.empty()) return;
        while ((int)cur.size() < W) cur.push_back(WarpWork{-1, 0, 0, 0});
        L.work.insert(L.work.end(), cur.begin(), cur.end());
        L.item_round0.push_back((int32_t)(L.work.size() / W));
        cur.clear();
    };
    for (int32_t t = 0; t < T; ++t) {
        if (seg_w[t] < kWarp) {
            // a shared tile is one warp's work; `first` also carries the segment width and the number of templates
            if (seg_idx[t] != 0) continue;
            if ((int)cur.size() + 1 > W) flush();
            const int first = (int)cur.size();
            cur.push_back(WarpWork{(int32_t)L.tile_begin[t], t, first | (seg_w[t] << 8) | (tile_nseg[(size_t)L.tile_begin[t]] << 16), 1});
            continue;
        }
        const int64_t nt = (off[t + 1] - off[t] + per_tile - 1) / per_tile;
        if (nt <= W) {
            if ((int64_t)cur.size() + nt > W) flush();
            const int first = (int)cur.size();
            for (int64_t i = 0; i < nt; ++i)
                cur.push_back(WarpWork{(int32_t)(L.tile_begin[t] + i), t, first, (int32_t)nt});
        } else {
            flush();
            for (int64_t i0 = 0; i0 < nt; i0 += W) {
                const int cnt = (int)std::min<int64_t>(W, nt - i0);
                for (int i = 0; i < W; ++i)
                    L.work.push_back(i < cnt ? WarpWork{(int32_t)(L.tile_begin[t] + i0 + i), t, 0, cnt}
                                             : WarpWork{-1, 0, 0, 0});
            }
            L.item_round0.push_back((int32_t)(L.work.size() / W));
        }
    }
    flush();
    L.coef.assign((size_t)L.n_tiles * 5 * per_tile, 0.f);
    for (int64_t tile = 0; tile < L.n_tiles; ++tile) {
        float* rec = L.coef.data() + (size_t)tile * 5 * per_tile;
        for (int64_t r = 0; r < per_tile; ++r) {
            const int64_t sl = tile * per_tile + r;
            rec[r] = L.ar[(size_t)sl];
            rec[per_tile + r] = L.ai[(size_t)sl];
            rec[2 * per_tile + 2 * r] = L.b[(size_t)(2 * sl)];
            rec[2 * per_tile + 2 * r + 1] = L.b[(size_t)(2 * sl + 1)];
            int32_t dl = L.dly[(size_t)sl];
            float bits;
            static_assert(sizeof(bits) == sizeof(dl), "delay is stored as int bits in a float slot");
            memcpy(&bits, &dl, sizeof(bits));
            rec[4 * per_tile + r] = bits;
        }
    }
    // Named per-template barriers are only safe when a warp position always belongs to the same group shape:
    // otherwise a fast warp could enter a hardware barrier that a slower group of another shape still uses.
    {
        std::vector<int32_t> first(W, -1), count(W, -1);
        if (L.segmented) L.uniform_groups = false;      // shared tiles store their sums themselves, behind CTA-wide barriers
        for (size_t i = 0; i < L.work.size(); ++i) {
            const WarpWork& w = L.work[i];
            if (w.tile < 0) continue;
            const int pos = (int)(i % (size_t)W);
            if (!L.uniform_groups) break;
            if (first[pos] < 0) { first[pos] = w.first; count[pos] = w.count; }
            else if (first[pos] != w.first || count[pos] != w.count) { L.uniform_groups = false; break; }
        }
        L.canon.assign((size_t)2 * W, 0);
        for (int w = 0; w < W; ++w) {
            L.canon[2 * w] = L.uniform_groups ? first[w] : -1;
            L.canon[2 * w + 1] = L.uniform_groups && first[w] >= 0 ? count[w] : 0;
        }
    }
    return L;
}

}  // namespace spiir
