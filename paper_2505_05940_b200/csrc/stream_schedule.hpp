// stream_schedule.hpp -- host-side layout of the STREAMING tensor-core vK kernel (vk_stream.cuh; DESIGN.md "Kernels /
// vk_stream"): small and medium batches on a tensor whose bf16 hi / lo copy does not fit the shared memory of the GPU
// (C4: N_q = 400, N_phi = 200 -> 45 MB).  No oracle code, no device code.
//
// Per time step t[(n,k)][b] = sum_r H^n[k][r] q[b][r] (Eq. 9 in one pass, C eliminated by PAPER.md:283) is the GEMM
//     D[(n,k)][b] = A[(n,k)][r] * Q[b][r]^T     M = 128 rows k of one k block for one in-plane mode n (a "tile"),
//                                               N = the samples (batch padded to 16, <= 64), K = the transverse modes r
// so a narrow batch does not waste a 128-row M tile: the rows of H are on M, the samples on N.  A (H as bf16 hi + lo, UMMA
// canonical K-major chunks of 128 rows x 16 K) is streamed from L2 by TMA every step; Q (q as bf16 hi + lo) is rebuilt in shared
// memory every step; D of all tiles of a CTA stays in TMEM (tiles x N columns <= 512) until eta is known.
//
// A CTA owns tiles of ONE k block (its threads' rows keep the running partial force in registers across the tiles) and, as owner,
// a few rows of that block for the update.  k blocks are contiguous ranges of the internal mode order aligned to its classes
// (the index parities of the sine-basis plate), at most 128 rows; K chunks of 16 never straddle two blocks; per tile only the K
// chunks with a non-zero are stored and multiplied.
#pragma once
#include <algorithm>
#include <cstdint>
#include <vector>
#include "mma_schedule.hpp"   // bf16 helpers, umma_chunk_off

namespace modal_host {

constexpr int ST_ROWS = 128;         // rows of a tile
constexpr int ST_BCH_MAX = 16;       // most K chunks of q one CTA keeps as B operand
constexpr int ST_TILES_MAX = 16;     // most tiles of one CTA (TMEM: tiles * NB <= 512)
constexpr int ST_NKB_MAX = 8;        // most k blocks
constexpr int ST_SENT_MAX = 256;     // most owner CTAs whose q one CTA waits for

struct StreamBlock { int k0, nb, koff; };

struct StreamTile { int n, jb, nch; size_t a_off; std::vector<int> chunks; };   // a_off: bytes into the A stream

struct StreamLayout {
    int n_q = 0, n_phi = 0, NB = 0, G = 0;
    int NKB = 0, KC = 0;                             // k blocks, K chunks of the operand axis
    std::vector<StreamBlock> blocks;
    std::vector<StreamTile> tiles;                   // in CTA order
    std::vector<int> cta_tile0, cta_ntiles, cta_block;   // [G]
    std::vector<int> cta_bch;                        // [G][ST_BCH_MAX]: global K chunks of the CTA's B operand (-1: unused)
    std::vector<int> cta_nbch;                       // [G]
    std::vector<int> cta_row0, cta_rows;             // [G]: rows of the CTA's block it owns for the update
    std::vector<int> blk_cta0, blk_nctas;            // [NKB]: the CTAs of a block are contiguous
    std::vector<int> tile_of;                        // [n_phi][NKB]: tile index of (n, block) or -1
    int tiles_max = 0, rows_max = 0, bch_max = 0, nch_max = 0;
    size_t a_bytes = 0;
    // device tables, ints.  Per CTA: [0] tile0 [1] ntiles [2] block [3] nbch [4] row0 [5] rows [6..] bch[ST_BCH_MAX] (chunk | valid << 16)
    // per tile (global): n, nch, a_off / 8192 (chunk units), mask of the k blocks with a tile of mode n (the contributors to G_n),
    // then nch x (B slot of the chunk)  -- stride TILE_STRIDE
    static constexpr int CTA_STRIDE = 6 + ST_BCH_MAX + 1 + ST_SENT_MAX;   // ... [22] sentinels [23..] operand positions: first row of every owner CTA this CTA reads q from
    int TILE_STRIDE = 0;
    std::vector<int> cta_tab, tile_tab;
};

// nz(n, k_int, r_int): H^n[k][r] != 0.  class_start: classes of the internal order (ncls + 1 entries).
template <class NZ>
inline bool stream_layout(int n_q, int n_phi, int sm, int NB, const std::vector<int> &class_start, NZ nz, StreamLayout &L)
{
    L = StreamLayout();
    L.n_q = n_q; L.n_phi = n_phi; L.NB = NB;
    // k blocks: classes cut into parts of <= 128 rows
    int koff = 0;
    for (size_t c = 0; c + 1 < class_start.size(); ++c) {
        const int k0 = class_start[c], len = class_start[c + 1] - k0;
        if (len <= 0) continue;
        const int parts = (len + ST_ROWS - 1) / ST_ROWS;
        for (int p = 0; p < parts; ++p) {
            const int a = k0 + (int)((long long)len * p / parts), b = k0 + (int)((long long)len * (p + 1) / parts);
            L.blocks.push_back({a, b - a, koff});
            koff += (b - a + 15) / 16 * 16;
        }
    }
    L.NKB = (int)L.blocks.size(); L.KC = koff / 16;
    if (L.NKB > ST_NKB_MAX || (NB != 16 && NB != 32 && NB != 64)) return false;
    std::vector<int> kop(koff, -1);
    for (const StreamBlock &b : L.blocks) for (int x = 0; x < b.nb; ++x) kop[b.koff + x] = b.k0 + x;
    // tiles and their K chunks
    std::vector<std::vector<StreamTile>> per_block(L.NKB);
    for (int jb = 0; jb < L.NKB; ++jb)
        for (int n = 0; n < n_phi; ++n) {
            StreamTile t; t.n = n; t.jb = jb; t.a_off = 0;
            for (int kc = 0; kc < L.KC; ++kc) {
                bool any = false;
                for (int e = 0; e < 16 && !any; ++e) {
                    const int r = kop[kc * 16 + e];
                    if (r < 0) continue;
                    for (int kk = 0; kk < L.blocks[jb].nb && !any; ++kk) any = nz(n, L.blocks[jb].k0 + kk, r);
                }
                if (any) t.chunks.push_back(kc);
            }
            t.nch = (int)t.chunks.size();
            if (t.nch) per_block[jb].push_back(t);
        }
    // CTAs per block in proportion to the work (chunks); tiles sorted by chunk signature so that a CTA's tiles share q chunks
    long long total = 0;
    std::vector<long long> work(L.NKB, 0);
    for (int jb = 0; jb < L.NKB; ++jb) {
        std::stable_sort(per_block[jb].begin(), per_block[jb].end(), [](const StreamTile &a, const StreamTile &b) { return a.chunks < b.chunks; });
        for (const StreamTile &t : per_block[jb]) work[jb] += t.nch + 2;
        total += work[jb];
    }
    if (total == 0) return false;
    std::vector<int> nct(L.NKB, 0), cap(L.NKB, 0);
    int used = 0;
    for (int jb = 0; jb < L.NKB; ++jb) {                 // a CTA has at least one tile and owns at least one row of its block
        cap[jb] = std::min((int)per_block[jb].size(), L.blocks[jb].nb);
        nct[jb] = std::min(cap[jb], std::max(1, (int)((long long)sm * work[jb] / total)));
        used += nct[jb];
    }
    while (used > sm) { int j = (int)(std::max_element(nct.begin(), nct.end()) - nct.begin()); --nct[j]; --used; }
    while (used < sm) {      // spare CTAs to the block with the most work per CTA
        int best = -1; double bw = 0;
        for (int jb = 0; jb < L.NKB; ++jb) if (nct[jb] && (double)work[jb] / nct[jb] > bw && nct[jb] < cap[jb]) { bw = (double)work[jb] / nct[jb]; best = jb; }
        if (best < 0) break;
        ++nct[best]; ++used;
    }
    L.G = used;
    L.blk_cta0.assign(L.NKB, 0); L.blk_nctas = nct;
    L.tile_of.assign((size_t)n_phi * L.NKB, -1);
    const int tiles_cap = std::min(ST_TILES_MAX, 512 / (NB <= 32 ? 2 * NB : NB));      // TMEM columns: 2 NB per tile when NB <= 32 (dual accumulator halves)
    int cta = 0;
    for (int jb = 0; jb < L.NKB; ++jb) {
        L.blk_cta0[jb] = cta;
        const std::vector<StreamTile> &ts = per_block[jb];
        double acc = 0; size_t i = 0;
        for (int x = 0; x < nct[jb]; ++x, ++cta) {
            const double goal = (double)work[jb] * (x + 1) / nct[jb];
            const int t0 = (int)L.tiles.size();
            std::vector<int> bch;
            while (i < ts.size()) {
                const bool must = (int)L.tiles.size() == t0;                                              // every CTA has a tile ...
                const bool can = ts.size() - i - 1 >= (size_t)(nct[jb] - 1 - x);                          // ... and leaves one for every later CTA
                const bool want = acc + 0.5 * (ts[i].nch + 2) < goal || x == nct[jb] - 1;
                if (!(must || (want && can))) break;
                L.tiles.push_back(ts[i]);
                for (int kc : ts[i].chunks) if (std::find(bch.begin(), bch.end(), kc) == bch.end()) bch.push_back(kc);
                acc += ts[i].nch + 2; ++i;
            }
            const int nt = (int)L.tiles.size() - t0;
            if (nt > tiles_cap || nt == 0 || (int)bch.size() > ST_BCH_MAX) return false;
            std::sort(bch.begin(), bch.end());
            L.cta_tile0.push_back(t0); L.cta_ntiles.push_back(nt); L.cta_block.push_back(jb);
            L.cta_nbch.push_back((int)bch.size());
            for (int u = 0; u < ST_BCH_MAX; ++u) L.cta_bch.push_back(u < (int)bch.size() ? bch[u] : -1);
            // owned rows of the block: an even share
            const int r0 = (int)((long long)L.blocks[jb].nb * x / nct[jb]), r1 = (int)((long long)L.blocks[jb].nb * (x + 1) / nct[jb]);
            if (r1 <= r0) return false;            // every CTA owns a row: its owners are a link of the step-to-step dependency chain
            L.cta_row0.push_back(r0); L.cta_rows.push_back(r1 - r0);
            L.tiles_max = std::max(L.tiles_max, nt); L.rows_max = std::max(L.rows_max, r1 - r0); L.bch_max = std::max(L.bch_max, (int)bch.size());
        }
    }
    // A stream offsets, tables
    size_t off = 0;
    for (size_t t = 0; t < L.tiles.size(); ++t) {
        L.tiles[t].a_off = off; off += (size_t)L.tiles[t].nch * 8192;
        L.tile_of[(size_t)L.tiles[t].n * L.NKB + L.tiles[t].jb] = (int)t;
        L.nch_max = std::max(L.nch_max, L.tiles[t].nch);
    }
    L.a_bytes = off;
    L.TILE_STRIDE = 4 + L.nch_max;
    L.cta_tab.assign((size_t)L.G * StreamLayout::CTA_STRIDE, 0);
    auto owner_first_row = [&](int jb, int row) {       // first row of the CTA of block jb that owns `row` (rows are cut as nb * x / nct)
        const int nb = L.blocks[jb].nb, nct = L.blk_nctas[jb];
        int x = (int)(((long long)row * nct) / nb);
        while (x + 1 < nct && (int)((long long)nb * (x + 1) / nct) <= row) ++x;
        while (x > 0 && (int)((long long)nb * x / nct) > row) --x;
        return (int)((long long)nb * x / nct);
    };
    for (int c = 0; c < L.G; ++c) {
        int *p = &L.cta_tab[(size_t)c * StreamLayout::CTA_STRIDE];
        p[0] = L.cta_tile0[c]; p[1] = L.cta_ntiles[c]; p[2] = L.cta_block[c]; p[3] = L.cta_nbch[c]; p[4] = L.cta_row0[c]; p[5] = L.cta_rows[c];
        std::vector<int> sent;
        auto need = [&](int kop) {
            for (int jb = 0; jb < L.NKB; ++jb) {
                const StreamBlock &b = L.blocks[jb];
                if (kop < b.koff || kop >= b.koff + b.nb) continue;
                const int s = b.koff + owner_first_row(jb, kop - b.koff);
                if (std::find(sent.begin(), sent.end(), s) == sent.end()) sent.push_back(s);
            }
        };
        for (int u = 0; u < ST_BCH_MAX; ++u) {       // chunk | valid K positions << 16 (the padding behind a block's last mode is never published)
            const int kc = L.cta_bch[(size_t)c * ST_BCH_MAX + u];
            int valid = 0;
            if (kc >= 0) for (const StreamBlock &b : L.blocks) if (kc * 16 >= b.koff && kc * 16 < b.koff + b.nb) valid = std::min(16, b.koff + b.nb - kc * 16);
            p[6 + u] = kc < 0 ? 0 : (kc | valid << 16);
            for (int e = 0; e < valid; ++e) need(kc * 16 + e);
        }
        for (int x = 0; x < L.blocks[L.cta_block[c]].nb; ++x) need(L.blocks[L.cta_block[c]].koff + x);
        if ((int)sent.size() > ST_SENT_MAX) return false;
        p[6 + ST_BCH_MAX] = (int)sent.size();
        for (size_t x = 0; x < sent.size(); ++x) p[7 + ST_BCH_MAX + x] = sent[x];
    }
    L.tile_tab.assign(L.tiles.size() * L.TILE_STRIDE, 0);
    for (int c = 0; c < L.G; ++c)
        for (int x = 0; x < L.cta_ntiles[c]; ++x) {
            const int t = L.cta_tile0[c] + x;
            int *p = &L.tile_tab[(size_t)t * L.TILE_STRIDE];
            p[0] = L.tiles[t].n; p[1] = L.tiles[t].nch; p[2] = (int)(L.tiles[t].a_off / 8192);
            for (int jb = 0; jb < L.NKB; ++jb) if (L.tile_of[(size_t)L.tiles[t].n * L.NKB + jb] >= 0) p[3] |= 1 << jb;
            for (int u = 0; u < L.tiles[t].nch; ++u) {
                const int *b = &L.cta_bch[(size_t)c * ST_BCH_MAX];
                p[4 + u] = (int)(std::find(b, b + ST_BCH_MAX, L.tiles[t].chunks[u]) - b);
            }
        }
    return true;
}

// A stream: per tile its chunks, each 8 KiB = [hi: 128 rows x 16 K bf16, canonical layout][lo].  get(n, k_int, r_int) -> double.
template <class Get>
inline void pack_stream_A(const StreamLayout &L, Get get, std::vector<uint16_t> &A)
{
    A.assign(L.a_bytes / 2, 0);
    std::vector<int> kop(L.KC * 16, -1);
    for (const StreamBlock &b : L.blocks) for (int x = 0; x < b.nb; ++x) kop[b.koff + x] = b.k0 + x;
    for (const StreamTile &t : L.tiles)
        for (int u = 0; u < t.nch; ++u) {
            uint16_t *base = &A[(t.a_off + (size_t)u * 8192) / 2];
            for (int kk = 0; kk < L.blocks[t.jb].nb; ++kk)
                for (int e = 0; e < 16; ++e) {
                    const int r = kop[t.chunks[u] * 16 + e];
                    if (r < 0) continue;
                    const float v = (float)get(t.n, L.blocks[t.jb].k0 + kk, r);
                    if (v == 0.f) continue;
                    const uint16_t hi = bf16_rn(v), lo = bf16_rn(v - bf16_to_float(hi));
                    const int o = umma_chunk_off(kk, e);
                    base[o / 2] = hi; base[(4096 + o) / 2] = lo;
                }
        }
}

}  // namespace modal_host
