// sa_tc5_schedule.cu -- host-side static schedule of the prefill items of one call over the
// persistent CTAs of the tcgen05 kernel ("batch planning").
//
// The cost of an item (request, kv head, 256 packed rows) is its number of 128-key KV tiles: the
// causal work A_j of PAPER.md L313 cut into tiles.  A chunk of 2,048 tokens on a 24K prefix is
// 256 equal items: on 148 SMs a whole-item schedule runs two waves and idles 27 % of the second.
// A 512-token lookahead chunk ("dynamic chunks") is 64 items: 84 SMs would idle.
// So items are assigned greedily, in locality order, to the least-loaded CTA (what the hardware
// block scheduler would do), and an item that does not fit under the balanced makespan is cut
// along KV into parts (stream-K); a split item's parts are merged afterwards in KV order.
//
// Consequence for reproducibility (R17): the bits of a prefill row depend on the set
// of prefill requests of the call (through the cut points), never on decode rows or on physical
// pages; the same call always gives the same bits.
#include <algorithm>

#include "sa_internal.h"

namespace sa {

void tc5_schedule(const std::vector<ReqMeta> &pre, int G, int Hkv, int n_cta, Tc5Schedule *out) {
    out->cta_begin.assign(size_t(n_cta) + 1, 0);
    out->parts.clear();
    out->merges.clear();
    out->n_slots = 0;
    out->total_units = 0;
    out->makespan = 0;

    struct Item {
        int32_t req, g, tile, n_kv;
    };
    std::vector<Item> items;
    {
        size_t n_items = 0;
        for (const ReqMeta &r : pre) n_items += size_t(Hkv) * size_t((int64_t(r.q_len) * G + kTc5TileM - 1) / kTc5TileM);
        items.reserve(n_items);
    }
    for (size_t ri = 0; ri < pre.size(); ++ri) {
        const ReqMeta &r = pre[ri];
        const int64_t n_rows = int64_t(r.q_len) * G;
        const int n_tiles = int((n_rows + kTc5TileM - 1) / kTc5TileM);
        const int base_lim = r.kv_len - r.q_len;
        // locality order: the tiles of one (request, kv head) are adjacent, late (heavy) tiles first,
        // so CTAs that run at the same time stream the same K/V through L2
        for (int g = 0; g < Hkv; ++g)
            for (int tile = n_tiles - 1; tile >= 0; --tile) {
                const int64_t rho_last = int64_t(tile) * kTc5TileM + kTc5TileM - 1;
                const int tok_max = int(std::min<int64_t>(r.q_len - 1, rho_last / G));
                const int k_end = base_lim + tok_max + 1;
                const int n_kv = (k_end + kTc5KeysPerUnit - 1) / kTc5KeysPerUnit;
                items.push_back({int32_t(ri), g, tile, n_kv});
                out->total_units += n_kv;
            }
    }
    if (items.empty()) return;

    const int64_t F = kTc5FixedCost;
    int64_t T = (out->total_units + F * (int64_t(items.size()) + n_cta) + n_cta - 1) / n_cta;
    T = std::max<int64_t>(T, kTc5MinPart + F);

    // Min-heap of (load, cta): least loaded first, ties by CTA index (a total order: the top is unique, so the
    // schedule does not depend on the heap's internal layout).  The only update is "give the top more load".
    typedef std::pair<int64_t, int32_t> Load;
    std::vector<Load> heap(static_cast<size_t>(n_cta));
    for (int c = 0; c < n_cta; ++c) heap[size_t(c)] = Load(0, c);  // ascending: already a heap
    auto raise_top = [&heap, n_cta](int64_t new_load) {
        Load x(new_load, heap[0].second);
        int i = 0;
        for (;;) {
            int ch = 2 * i + 1;
            if (ch >= n_cta) break;
            if (ch + 1 < n_cta && heap[size_t(ch + 1)] < heap[size_t(ch)]) ++ch;
            if (!(heap[size_t(ch)] < x)) break;
            heap[size_t(i)] = heap[size_t(ch)];
            i = ch;
        }
        heap[size_t(i)] = x;
    };
    // parts in creation order; grouped by CTA afterwards with a stable counting sort (this runs on the host inside
    // every sa_mixed_attention call: no per-CTA vectors, no reallocation)
    std::vector<Tc5Part> flat;
    flat.reserve(items.size() + size_t(n_cta) + 8);
    std::vector<int32_t> per_cta_count(size_t(n_cta), 0);
    out->merges.reserve(size_t(n_cta) + 8);

    for (const Item &it : items) {
        int u = 0;
        int first_slot = out->n_slots, n_parts = 0;
        bool split = false;
        while (u < it.n_kv) {
            const Load top = heap[0];
            const int64_t cap = T - top.first - F;
            const int remaining = it.n_kv - u;
            int take;
            if (cap >= kTc5MinPart && remaining - cap < kTc5MinPart) {
                take = remaining;  // fits, or overshoots the makespan by less than a minimum part
            } else if (cap >= kTc5MinPart) {
                take = int(cap);
            } else if (cap >= remaining) {
                take = remaining;
            } else {
                T += kTc5MinPart;  // every CTA is (nearly) full: raise the makespan a little and retry
                continue;
            }
            Tc5Part p;
            p.req = it.req;
            p.g = it.g;
            p.tile = it.tile;
            p.u0 = u;
            p.u1 = u + take;
            p.n_kv = it.n_kv;
            p.cta = top.second;
            split = split || take < it.n_kv;
            p.slot = split ? out->n_slots++ : -1;
            flat.push_back(p);
            ++per_cta_count[size_t(top.second)];
            raise_top(top.first + take + F);
            u += take;
            ++n_parts;
        }
        if (split) {
            Tc5Merge m{};
            m.req = it.req;
            m.g = it.g;
            m.tile = it.tile;
            m.slot0 = first_slot;
            m.n_parts = n_parts;
            out->merges.push_back(m);
        }
    }
    int32_t run = 0;
    for (int c = 0; c < n_cta; ++c) {
        out->cta_begin[size_t(c)] = run;
        run += per_cta_count[size_t(c)];
    }
    out->cta_begin[size_t(n_cta)] = run;
    out->parts.resize(flat.size());
    std::vector<int32_t> cursor(out->cta_begin.begin(), out->cta_begin.end() - 1);
    std::vector<int64_t> load(size_t(n_cta), 0);
    for (const Tc5Part &p : flat) {  // creation order within a CTA = execution order
        out->parts[size_t(cursor[size_t(p.cta)]++)] = p;
        load[size_t(p.cta)] += p.u1 - p.u0 + F;
    }
    for (int c = 0; c < n_cta; ++c) out->makespan = std::max(out->makespan, load[size_t(c)]);
}

}  // namespace sa
