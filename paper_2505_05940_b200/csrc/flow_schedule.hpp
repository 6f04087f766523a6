// flow_schedule.hpp -- host-side work schedule and tile layout of the vK "flow" kernel
// (vk_flow.cuh).  No oracle code, no device code.
//
// Tile layout ("flow tiles").  H^n (symmetric, Eq. 10) is cut into 16x16 tiles
// of the zero-padded matrix; only tiles (I,J), J <= I are stored, in the order
//     n-major, then I, then J           (global tile index  n*tpn + I(I+1)/2 + J).
// In diagonal tiles the strict upper part is zero and the diagonal is halved, so that the row pass
// plus the transposed column pass over the stored tiles give exactly H^n q.  Inside a tile the 256
// floats are ordered for the warp that consumes it: lane l = (half = l>>4, j = l&15) owns column j
// of rows half*8 .. half*8+7; element e of that lane sits at float (e>>2)*128 + l*4 + (e&3), i.e.
// the tile is two conflict-free LDS.128 per lane.
#pragma once
#include <algorithm>
#include <cstdint>
#include <vector>

namespace modal_host {

constexpr int FT = 16;              // tile edge
constexpr int FT_FLOATS = 256;      // floats per tile (1 KiB)

inline int flow_nt(int n_q) { return (n_q + FT - 1) / FT; }
inline int flow_tiles_per_n(int n_q) { const int nt = flow_nt(n_q); return nt * (nt + 1) / 2; }
inline int flow_padded_nq(int n_q) { return flow_nt(n_q) * FT; }
inline int flow_elem(int row_in_tile, int col_in_tile)
{
    const int half = row_in_tile >> 3, e = row_in_tile & 7, lane = half * 16 + col_in_tile;
    return (e >> 2) * 128 + lane * 4 + (e & 3);
}

template <class Get>   // Get(n,p,q) -> double
inline void pack_flow_tiles(int n_q, int n_phi, Get get, std::vector<float> &Hf)
{
    const int nt = flow_nt(n_q), tpn = nt * (nt + 1) / 2;
    Hf.assign((size_t)n_phi * tpn * FT_FLOATS, 0.f);
    for (int n = 0; n < n_phi; ++n)
        for (int I = 0; I < nt; ++I)
            for (int J = 0; J <= I; ++J) {
                float *t = &Hf[((size_t)n * tpn + I * (I + 1) / 2 + J) * FT_FLOATS];
                for (int i = 0; i < FT; ++i)
                    for (int j = 0; j < FT; ++j) {
                        const int p = I * FT + i, q = J * FT + j;
                        if (p >= n_q || q >= n_q || q > p) continue;
                        const double v = get(n, p, q);
                        t[flow_elem(i, j)] = (float)(p == q ? 0.5 * v : v);
                    }
            }
}

// inverse of pack_flow_tiles: the fp32 values the device holds, as a full symmetric fp64 tensor
inline void unpack_flow_tiles(int n_q, int n_phi, const std::vector<float> &Hf, double *H)
{
    const int nt = flow_nt(n_q), tpn = nt * (nt + 1) / 2;
    for (int n = 0; n < n_phi; ++n)
        for (int p = 0; p < n_q; ++p)
            for (int q = 0; q <= p; ++q) {
                const int I = p / FT, J = q / FT;
                const float t = Hf[((size_t)n * tpn + I * (I + 1) / 2 + J) * FT_FLOATS + flow_elem(p % FT, q % FT)];
                const double v = p == q ? 2.0 * (double)t : (double)t;
                H[((size_t)n * n_q + p) * n_q + q] = v;
                H[((size_t)n * n_q + q) * n_q + p] = v;
            }
}

// ---------------------------------------------------------------------------------------------
// Schedule.  A *unit* is a run of <= slot_tiles consecutive tiles of one tile row (n, I, J0..);
// it is the granule a consumer warp processes and the granule the TMA producer streams.  The
// units, in global tile order, are cut into G contiguous ranges of equal cost, one per CTA of a
// team (rank 0..G-1).  An in-plane mode n whose units fall into several CTAs is *shared*: the
// sharers exchange their partial G_n (vk_flow.cuh, phase B1).
//
// Per-CTA table blob (ints), consumed by the kernel from shared memory:
//   [0] U units  [1] R resident units  [2] NLOC pieces  [3] E list entries  [4] slice0  [5] slice_len
//   [6] resident tiles  [7] reserved
//   units   [U][4] : {nloc | I<<8 | ntiles<<16 , J0, tpoff, gtile0}     (gtile0: global tile index)
//   ltile   [U]    : tile offset inside the resident area (units < R)
//   pieces  [NLOC][4] : {n, first sharer rank, number of sharers, my slot}
//   pu      [NLOC+1]  : unit range of each piece
//   kb_ptr  [nb+1], kb_list [E] : per 16-mode block K, the tp groups that contribute to f_k, k in K:
//                                 entry = tp offset (floats) | nloc << 24
// ---------------------------------------------------------------------------------------------
struct FlowSchedule {
    int G = 1, NW = 16, slot_tiles = 8;
    int nt = 0, tpn = 0, NQP = 0, nb = 0;
    int U_max = 0, tp_max = 0, E_max = 0, NLOC_MAX = 0, tiles_max = 0, slice_max = 0, MS = 1;
    int stride = 0;                       // ints per CTA blob
    std::vector<int> blob;                // [G][stride]
    // offsets inside a blob, identical for every CTA (sized by the maxima)
    int off_units = 8, off_ltile = 0, off_pieces = 0, off_pu = 0, off_kbptr = 0, off_kblist = 0;
    std::vector<int> cta_tiles;           // [G] tiles per CTA
};

// tile_nz: optional [n_phi * tpn] flags, 0 = the tile holds only zeros and is left out of the schedule (it is never read:
// with the modes grouped by index parity ~70 % of the tiles of the sine-basis tensor vanish).
inline FlowSchedule build_flow_schedule(int n_q, int n_phi, int G, int NW, int slot_tiles, const std::vector<uint8_t> *tile_nz = nullptr)
{
    FlowSchedule s;
    s.G = G; s.NW = NW; s.slot_tiles = slot_tiles;
    const int nt = flow_nt(n_q), tpn = nt * (nt + 1) / 2;
    s.nt = nt; s.tpn = tpn; s.NQP = nt * FT; s.nb = nt;
    struct Atom { int n, I, J0, ntl; };
    std::vector<Atom> atoms;
    for (int n = 0; n < n_phi; ++n)
        for (int I = 0; I < nt; ++I) {
            // maximal runs of non-zero tiles of this tile row, each cut into parts of <= slot_tiles tiles
            for (int J = 0; J <= I;) {
                auto nz = [&](int jj) { return !tile_nz || (*tile_nz)[(size_t)n * tpn + I * (I + 1) / 2 + jj] != 0; };
                if (!nz(J)) { ++J; continue; }
                int e = J;
                while (e <= I && nz(e)) ++e;
                const int len = e - J, parts = (len + slot_tiles - 1) / slot_tiles;
                for (int p = 0, j = J; p < parts; ++p) {
                    const int l = len / parts + (p < len % parts ? 1 : 0);
                    atoms.push_back({n, I, j, l});
                    j += l;
                }
                J = e;
            }
        }
    const double unit_overhead = 1.5;     // tile-equivalents of per-unit epilogue work
    double total = 0;
    for (const Atom &a : atoms) total += a.ntl + unit_overhead;
    std::vector<int> first(G + 1, 0);
    // (a) whole in-plane modes per CTA (no mode is shared, so phase B1 needs no exchange): longest-processing-time
    //     assignment of the modes; taken when its most loaded CTA stays within 10 % of the ideal share
    bool whole_modes = false;
    if (G > 1 && G <= n_phi) {
        std::vector<double> cost(n_phi, 0.0);
        for (const Atom &a : atoms) cost[a.n] += a.ntl + unit_overhead;
        std::vector<int> order(n_phi);
        for (int n = 0; n < n_phi; ++n) order[n] = n;
        std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return cost[x] > cost[y]; });
        std::vector<double> load(G, 0.0);
        std::vector<int> owner(n_phi, 0);
        for (int n : order) {
            const int c = (int)(std::min_element(load.begin(), load.end()) - load.begin());
            owner[n] = c; load[c] += cost[n];
        }
        if (*std::max_element(load.begin(), load.end()) <= 1.10 * total / G) {
            whole_modes = true;
            std::vector<Atom> sorted;
            sorted.reserve(atoms.size());
            for (int c = 0; c < G; ++c) {
                first[c] = (int)sorted.size();
                for (int n = 0; n < n_phi; ++n)
                    if (owner[n] == c)
                        for (const Atom &a : atoms) if (a.n == n) sorted.push_back(a);
            }
            first[G] = (int)sorted.size();
            atoms.swap(sorted);
        }
    }
    // (b) otherwise: contiguous partition of the units by cumulative cost (modes may be shared between CTAs)
    if (!whole_modes) {
        double acc = 0; int c = 1;
        for (size_t i = 0; i < atoms.size(); ++i) {
            const double mid = acc + 0.5 * (atoms[i].ntl + unit_overhead);
            while (c < G && mid >= total * c / G) first[c++] = (int)i;
            acc += atoms[i].ntl + unit_overhead;
        }
        while (c <= G) first[c++] = (int)atoms.size();
    }
    // sharers of each n: the CTAs that hold units of n, in rank order (idle CTAs in between hold none)
    std::vector<std::vector<int>> holders(n_phi);
    for (int c = 0; c < G; ++c)
        for (int i = first[c]; i < first[c + 1]; ++i)
            if (holders[atoms[i].n].empty() || holders[atoms[i].n].back() != c) holders[atoms[i].n].push_back(c);
    for (int n = 0; n < n_phi; ++n) s.MS = std::max(s.MS, (int)holders[n].size());
    // maxima
    s.cta_tiles.assign(G, 0);
    for (int c = 0; c < G; ++c) {
        int U = first[c + 1] - first[c], tiles = 0, nloc = 0, lastn = -1;
        for (int i = first[c]; i < first[c + 1]; ++i) {
            tiles += atoms[i].ntl;
            if (atoms[i].n != lastn) { ++nloc; lastn = atoms[i].n; }
        }
        s.cta_tiles[c] = tiles;
        s.U_max = std::max(s.U_max, U);
        s.tiles_max = std::max(s.tiles_max, tiles);
        s.tp_max = std::max(s.tp_max, (tiles + U) * FT);
        s.E_max = std::max(s.E_max, tiles + U);
        s.NLOC_MAX = std::max(s.NLOC_MAX, nloc);
    }
    s.slice_max = (s.NQP + G - 1) / G;
    s.off_units = 8;
    s.off_ltile = s.off_units + 4 * s.U_max;
    s.off_pieces = (s.off_ltile + s.U_max + 3) / 4 * 4;      // int4 reads: 16-byte aligned
    s.off_pu = s.off_pieces + 4 * s.NLOC_MAX;
    s.off_kbptr = s.off_pu + s.NLOC_MAX + 1;
    s.off_kblist = s.off_kbptr + s.nb + 1;
    s.stride = ((s.off_kblist + s.E_max + 3) / 4) * 4;
    s.blob.assign((size_t)G * s.stride, 0);
    for (int c = 0; c < G; ++c) {
        int *b = &s.blob[(size_t)c * s.stride];
        const int U = first[c + 1] - first[c];
        int nloc = -1, lastn = -1, tp = 0, lt = 0;
        std::vector<std::vector<int>> lists(s.nb);
        for (int u = 0; u < U; ++u) {
            const Atom &a = atoms[first[c] + u];
            if (a.n != lastn) {
                ++nloc; lastn = a.n;
                int *p = b + s.off_pieces + 4 * nloc;
                const std::vector<int> &hs = holders[a.n];
                p[0] = a.n; p[1] = hs.front(); p[2] = (int)hs.size();
                p[3] = (int)(std::find(hs.begin(), hs.end(), c) - hs.begin());
                b[s.off_pu + nloc] = u;
            }
            int *w = b + s.off_units + 4 * u;
            w[0] = nloc | (a.I << 8) | (a.ntl << 16);
            w[1] = a.J0; w[2] = tp; w[3] = a.n * tpn + a.I * (a.I + 1) / 2 + a.J0;
            b[s.off_ltile + u] = lt;
            for (int t = 0; t < a.ntl; ++t) lists[a.J0 + t].push_back((tp + t * FT) | (nloc << 24));   // column groups
            lists[a.I].push_back((tp + a.ntl * FT) | (nloc << 24));                                    // row group
            tp += (a.ntl + 1) * FT;
            lt += a.ntl;
        }
        b[s.off_pu + nloc + 1] = U;
        int e = 0;
        for (int K = 0; K < s.nb; ++K) {
            b[s.off_kbptr + K] = e;
            for (int v : lists[K]) b[s.off_kblist + e++] = v;
        }
        b[s.off_kbptr + s.nb] = e;
        b[0] = U; b[1] = U; b[2] = nloc + 1; b[3] = e;
        b[4] = (int)((long long)s.NQP * c / G);
        b[5] = (int)((long long)s.NQP * (c + 1) / G) - b[4];
        b[6] = lt; b[7] = 0;
    }
    return s;
}

// Set the number of resident units of every CTA to the longest prefix that fits `cap_tiles`
// tiles of shared memory; returns the largest number of streamed units of any CTA.
inline int flow_set_residency(FlowSchedule &s, int cap_tiles)
{
    int smax = 0;
    for (int c = 0; c < s.G; ++c) {
        int *b = &s.blob[(size_t)c * s.stride];
        const int U = b[0];
        int R = 0, tiles = 0;
        while (R < U) {
            const int ntl = (b[s.off_units + 4 * R] >> 16) & 0xff;
            if (tiles + ntl > cap_tiles) break;
            tiles += ntl; ++R;
        }
        b[1] = R; b[6] = tiles;
        smax = std::max(smax, U - R);
    }
    return smax;
}

}  // namespace modal_host
