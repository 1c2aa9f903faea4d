// tiler.cu -- S:8(a) A11: out-of-core window tiling.
//
// the edge arrays are cut into W row-aligned windows; a tile is a (hub window h, search
// window c) pair; the tuple rooted at edge (i,j) is processed in the one tile with i in h and j in c,
// and spokes whose row is not resident are skipped with one integer compare.  Here the windows live
// in pinned host memory and are streamed through a small cache of device buffers on a copy stream,
// so that the upload of the next tile's windows overlaps the enumeration of the current tile.
// Tiles whose search window holds no spoke of the hub window (known from the build) are not visited:
// with labels in cell order a hub window only reaches a few search windows.
#include "internal.cuh"

#include <algorithm>

namespace {

struct Slot {
    DevBuf<int32_t> idx;
    DevBuf<uint8_t> bin, pix;
    DevBuf<uint8_t> dense;         // dense cell-block rows of window `dense_wid`, expanded on the device from idx/bin
    int dense_wid = -1;
    int wid = -1;
    cudaEvent_t ready = nullptr, done = nullptr;
    uint64_t stamp = 0;
};

}  // namespace

// window buffers that fit under the cap (each: the window's CSR arrays, plus its dense rows when asked for)
int gr_tiler_slots(const gramsci_graph *g, bool need_pix, bool need_dense)
{
    const int W = (int)g->windows.size();
    const uint64_t bpe = 5 + ((g->has_pix && need_pix) ? 1 : 0);
    int64_t maxlen = 0, maxdense = 0;
    for (auto &w : g->windows) { maxlen = std::max(maxlen, w.e_hi - w.e_lo); maxdense = std::max(maxdense, w.d_hi - w.d_lo); }
    if (!need_dense) maxdense = 0;
    const int K = (int)std::min<uint64_t>((uint64_t)W, g->cap_bytes / std::max<uint64_t>(1, (uint64_t)maxlen * bpe + (uint64_t)maxdense));
    return std::min(K, 8);
}

void gr_for_each_tile(gramsci_graph *g, bool need_pix, bool hub_only, gr_tile_fn fn, void *user, bool need_dense, bool pair_search)
{
    cudaStream_t st = g->stream;
    GrView v;
    v.ptr = g->ptr.p;
    v.order = g->order.p;
    v.w = g->w.p;
    v.hub_stride = g->hub_stride;
    v.shard_count = g->shard_count;
    v.shard_index = g->shard_index;
    v.dense = g->dn.bytes.p;
    v.d0 = 0;
    v.dense_span = g->dn.total;
    if (!g->ooc) {
        v.idx_h = v.idx_c = g->idx.p;
        v.bin_h = v.bin_c = g->bin.p;
        v.pix_h = v.pix_c = g->has_pix ? g->pix.p : nullptr;
        v.e0_h = v.e0_c = 0;
        v.c_lo = 0;
        v.c_hi = (int32_t)g->n;
        v.h_lo = std::max(0, g->hub_lo);
        v.h_hi = (int32_t)std::min<int64_t>(g->n, g->hub_hi);
        v.win_h = 0;
        v.idx_c2 = v.idx_c; v.bin_c2 = v.bin_c; v.e0_c2 = 0;
        v.c2_lo = 0; v.c2_hi = (int32_t)g->n;
        v.s_lo = g->spatial ? v.h_lo : 0;
        v.s_hi = g->spatial ? v.h_hi : (int32_t)g->n;
        if (v.h_hi > v.h_lo) fn(g, v, user, st);
        return;
    }

    const int W = (int)g->windows.size();
    const uint64_t bpe = 5 + (g->has_pix ? 1 : 0);
    int64_t maxlen = 0, maxdense = 0;
    for (auto &w : g->windows) { maxlen = std::max(maxlen, w.e_hi - w.e_lo); maxdense = std::max(maxdense, w.d_hi - w.d_lo); }
    if (!need_dense) maxdense = 0;
    const int K = gr_tiler_slots(g, need_pix, need_dense);
    if (pair_search && K < std::min(3, W))      // (two windows: every tile touches at most two)
        GR_FAIL(GRAMSCI_ENOMEM, "device_mem_cap_bytes too small for three windows of %lld edges (4pCF tiles, P:159)", (long long)maxlen);
    if (K < (hub_only ? 1 : 2)) GR_FAIL(GRAMSCI_ENOMEM, "device_mem_cap_bytes too small for two windows of %lld edges", (long long)maxlen);

    std::vector<Slot> slots(K);
    cudaStream_t cs = nullptr;
    GR_CUDA(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
    struct Cleanup {
        std::vector<Slot> &s; cudaStream_t cs;
        ~Cleanup() {
            cudaStreamSynchronize(cs);
            for (auto &x : s) { if (x.ready) cudaEventDestroy(x.ready); if (x.done) cudaEventDestroy(x.done); }
            cudaStreamDestroy(cs);
        }
    } cleanup{slots, cs};
    for (auto &s : slots) {
        s.idx.alloc((size_t)maxlen + 64);
        s.bin.alloc((size_t)maxlen + 64);
        if (g->has_pix && need_pix) s.pix.alloc((size_t)maxlen + 64);
        if (need_dense) s.dense.alloc((size_t)maxdense + 64);
        GR_CUDA(cudaEventCreateWithFlags(&s.ready, cudaEventDisableTiming));
        GR_CUDA(cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming));
    }
    // the window buffers are stream-ordered allocations on `st`: the copy stream may touch them only after
    // that point of `st`
    {
        cudaEvent_t ev;
        GR_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        GR_CUDA(cudaEventRecord(ev, st));
        GR_CUDA(cudaStreamWaitEvent(cs, ev, 0));
        GR_CUDA(cudaEventDestroy(ev));
    }
    uint64_t clock = 0;

    // bring window `wid` into a slot (cache hit: no copy); never evicts a slot whose bit is set in `protect`
    // the dense rows of the window in slot k (search windows of the gather kernel): memset + scatter on the copy stream,
    // after the window's CSR has arrived
    auto expand = [&](int k) {
        Slot &s = slots[k];
        if (!need_dense || s.dense_wid == s.wid) return;
        const GrWindow &w = g->windows[s.wid];
        if (s.dense_wid >= 0) GR_CUDA(cudaStreamWaitEvent(cs, s.done, 0));
        gr_dense_expand(g, w.row_lo, w.row_hi, s.idx.p, s.bin.p, w.e_lo, s.dense.p, w.d_lo, w.d_hi - w.d_lo, cs);
        GR_CUDA(cudaEventRecord(s.ready, cs));
        s.dense_wid = s.wid;
    };
    auto acquire = [&](int wid, unsigned protect, bool want_dense = false) -> int {
        for (int k = 0; k < K; ++k)
            if (slots[k].wid == wid) { slots[k].stamp = ++clock; if (want_dense) expand(k); return k; }
        int victim = -1;
        for (int k = 0; k < K; ++k) {
            if (protect & (1u << k)) continue;
            if (victim < 0 || slots[k].stamp < slots[victim].stamp) victim = k;
        }
        if (victim < 0) return -1;
        Slot &s = slots[victim];
        const GrWindow &w = g->windows[wid];
        const int64_t len = w.e_hi - w.e_lo;
        if (s.wid >= 0) GR_CUDA(cudaStreamWaitEvent(cs, s.done, 0));     // last kernel reading it has finished
        if (len > 0) {
            GR_CUDA(cudaMemcpyAsync(s.idx.p, w.h_idx, (size_t)len * 4, cudaMemcpyHostToDevice, cs));
            GR_CUDA(cudaMemcpyAsync(s.bin.p, w.h_bin, (size_t)len, cudaMemcpyHostToDevice, cs));
            if (g->has_pix && need_pix)
                GR_CUDA(cudaMemcpyAsync(s.pix.p, w.h_pix, (size_t)len, cudaMemcpyHostToDevice, cs));
            g->staged_bytes += (double)len * (5 + ((g->has_pix && need_pix) ? 1 : 0));
        }
        GR_CUDA(cudaEventRecord(s.ready, cs));
        s.wid = wid;
        s.stamp = ++clock;
        if (want_dense) expand(victim);
        return victim;
    };

    // tiles (h, c1, c2): 2pCF / 3pCF use c2 == c1; the 4pCF takes every pair c1 <= c2 of search windows the hub window
    // reaches (and, for c1 < c2, only if window c1 holds an edge into window c2 -- j1 ~ j2 is part of every tetrahedron)
    struct Tile { int h, c1, c2; };
    std::vector<Tile> tiles;
    auto needed = [&](int h, int c) { return g->need.empty() || g->need[(size_t)h * W + c]; };
    for (int h = 0; h < W; ++h) {
        if (std::min(g->windows[h].row_hi, g->hub_hi) <= std::max(g->windows[h].row_lo, g->hub_lo) && W > 1) continue;   // no owned hub
        if (hub_only) { tiles.push_back({h, h, h}); continue; }
        for (int c = 0; c < W; ++c) {
            if (!needed(h, c)) continue;
            if (!pair_search) { tiles.push_back({h, c, c}); continue; }
            for (int c2 = c; c2 < W; ++c2)
                if (needed(h, c2) && (c2 == c || needed(c, c2))) tiles.push_back({h, c, c2});
        }
    }
    const int T = (int)tiles.size();
    for (int t = 0; t < T; ++t) {
        const int a = acquire(tiles[t].h, 0);
        const int b = acquire(tiles[t].c1, 1u << a, need_dense);
        const int c = acquire(tiles[t].c2, (1u << a) | (1u << b), false);
        if (a < 0 || b < 0 || c < 0) GR_FAIL(GRAMSCI_ENOMEM, "window cache exhausted");
        GR_CUDA(cudaStreamWaitEvent(st, slots[a].ready, 0));
        GR_CUDA(cudaStreamWaitEvent(st, slots[b].ready, 0));
        GR_CUDA(cudaStreamWaitEvent(st, slots[c].ready, 0));
        const GrWindow &wh = g->windows[tiles[t].h], &wc = g->windows[tiles[t].c1], &wc2 = g->windows[tiles[t].c2];
        v.idx_h = slots[a].idx.p; v.bin_h = slots[a].bin.p; v.pix_h = slots[a].pix.p; v.e0_h = wh.e_lo;
        v.idx_c = slots[b].idx.p; v.bin_c = slots[b].bin.p; v.pix_c = slots[b].pix.p; v.e0_c = wc.e_lo;
        v.idx_c2 = slots[c].idx.p; v.bin_c2 = slots[c].bin.p; v.e0_c2 = wc2.e_lo;
        v.h_lo = std::max(wh.row_lo, g->hub_lo); v.h_hi = std::min(wh.row_hi, g->hub_hi);
        v.win_h = tiles[t].h;
        v.c_lo = wc.row_lo; v.c_hi = wc.row_hi;
        v.c2_lo = wc2.row_lo; v.c2_hi = wc2.row_hi;
        v.dense = need_dense ? slots[b].dense.p : nullptr;
        v.d0 = wc.d_lo;
        v.dense_span = wc.d_hi - wc.d_lo;
        if (g->spatial) { v.s_lo = v.h_lo; v.s_hi = v.h_hi; }
        else { v.s_lo = 0; v.s_hi = (int32_t)g->n; }
        if (v.h_hi > v.h_lo) fn(g, v, user, st);
        GR_CUDA(cudaEventRecord(slots[a].done, st));
        if (b != a) GR_CUDA(cudaEventRecord(slots[b].done, st));
        if (c != a && c != b) GR_CUDA(cudaEventRecord(slots[c].done, st));
        // prefetch the next tile's windows into slots the running tile does not use (copy stream)
        if (t + 1 < T) {
            unsigned protect = (1u << a) | (1u << b) | (1u << c);
            int s1 = acquire(tiles[t + 1].h, protect);
            if (s1 >= 0) {
                int s2 = acquire(tiles[t + 1].c1, protect | (1u << s1), need_dense);
                if (s2 >= 0 && tiles[t + 1].c2 != tiles[t + 1].c1) acquire(tiles[t + 1].c2, protect | (1u << s1) | (1u << s2), false);
            }
        }
    }
    GR_CUDA(cudaStreamSynchronize(st));
}
