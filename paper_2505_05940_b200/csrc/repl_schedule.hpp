// repl_schedule.hpp -- host-side layout of the REPLICATED-STATE von Karman kernel (vk_repl.cuh): one sample of a LARGE
// plate (C4: N_q = 400, N_phi = 200, BASELINE.json configs[1]) with ONE cross-CTA hop per time step.
// No oracle code, no device code.
//
// Every CTA keeps the whole fp64 state (bit-identical replicas) and owns whole in-plane modes n: t_n = H^n q, G_n = q . t_n,
// eta_n = s_n G_n and its part of the force sum_n eta_n t_n need no exchange (Eq. 9-11, C eliminated :283).  That
// takes H^n of the CTA's modes in shared memory, which only works because of two structural facts of the sine-basis plate
// (SURVEY.md 8(f) row 4): in the internal mode order (sorted by the index-parity class) H^n is a block matrix whose class a couples
// to ONE partner class b = a xor class(n), and H^n is symmetric.  So per mode only the blocks (a, b) with a <= b are stored, dense,
// fp32, rows padded to 16 bytes:
//   a <  b:  the block serves both t[a rows] += B q[b cols] (row sums) and t[b cols] += B^T q[a rows] (column sums)
//   a == b:  stored whole (it is symmetric itself); column sums only
// = 80 KiB per mode with off-diagonal blocks, 160 KiB per mode with diagonal blocks at C4: two, or one, per CTA.
//
// Work of a CTA per step: every thread owns one ITEM = (block, chunk of rows, quad of columns): nrows float4 loads.  The chunk
// length is chosen per CTA so that its items fill the 512 threads.  Partial column sums go to cpart[block][chunk][col], partial row
// sums to rpart[block][row][quad]; thread k then JOINS the partials of mode k for every mode of the CTA (fixed order).
#pragma once
#include <algorithm>
#include <cstdint>
#include <vector>

namespace modal_host {

constexpr int RP_THREADS = 512;
constexpr int RP_MAXM = 4;           // most in-plane modes of one CTA
constexpr int RP_MAXCLS = 8;         // most classes of the internal order
constexpr int RP_HDR = 16;           // ints of the per-CTA header
constexpr int RP_ITEM = 8;           // ints per item descriptor
constexpr int RP_JOIN = 4;           // ints per join descriptor
constexpr int RP_CTA_STRIDE = RP_HDR + RP_THREADS * RP_ITEM + RP_MAXM * RP_MAXCLS * RP_JOIN;

struct ReplBlock { int n, a, b; };   // mode, row class, column class (found with a <= b; a CTA may store it the other way round)

struct ReplLayout {
    int n_q = 0, n_phi = 0, G = 0, ncls = 0;
    std::vector<int> class_start;                 // ncls + 1
    std::vector<int> cta_nmodes, cta_modes;       // [G], [G][RP_MAXM]
    std::vector<size_t> cta_hoff;                 // [G] floats into Hp
    std::vector<int> cta_hfloats, cta_cp, cta_rp; // [G] floats of H, of cpart, of rpart
    int hfloats_max = 0, cp_max = 0, rp_max = 0, rows_max = 0, out_cta = 0;
    std::vector<float> Hp;                        // packed blocks, CTA after CTA
    // device table, RP_CTA_STRIDE ints per CTA:
    //   [0] hoff / 4 (float4 units into Hp)  [1] hfloats  [2] nmodes  [3] items  [4..8) mode ids
    //   items [t]: {hoff (floats into the CTA's H), ld | mode slot << 16, qa0, nrows, qb0, rp_off (-1: none), rp_stride, cp_off}
    //   joins [m][class]: {kind 0 none / 1 column sums / 2 row sums, base, count, stride of the partials (1) or pitch of a row (2)}
    std::vector<int> tab;
};

// H: dense [n_phi][n_q][n_q] in the internal order.  G: CTAs available.  cap_floats: shared memory for H + cpart + rpart.
inline bool repl_layout(int n_q, int n_phi, int G, size_t cap_floats, const std::vector<int> &class_start, const double *H, ReplLayout &L)
{
    L = ReplLayout();
    const int ncls = (int)class_start.size() - 1;
    if (n_q > RP_THREADS || ncls < 1 || ncls > RP_MAXCLS || G < 1) return false;
    L.n_q = n_q; L.n_phi = n_phi; L.G = G; L.ncls = ncls; L.class_start = class_start;
    auto len = [&](int c) { return class_start[c + 1] - class_start[c]; };
    auto ld = [&](int c) { return (len(c) + 3) & ~3; };
    // blocks of every mode; the stored set must reproduce H^n exactly (symmetry is checked here, not assumed)
    std::vector<std::vector<ReplBlock>> mblocks(n_phi);
    std::vector<size_t> cost(n_phi, 0);
    for (int n = 0; n < n_phi; ++n) {
        const double *Hn = H + (size_t)n * n_q * n_q;
        for (int a = 0; a < ncls; ++a)
            for (int b = 0; b < ncls; ++b) {
                bool any = false;
                for (int i = class_start[a]; i < class_start[a + 1] && !any; ++i)
                    for (int j = class_start[b]; j < class_start[b + 1]; ++j) if (Hn[(size_t)i * n_q + j] != 0.0) { any = true; break; }
                if (!any) continue;
                for (int i = class_start[a]; i < class_start[a + 1]; ++i)
                    for (int j = class_start[b]; j < class_start[b + 1]; ++j)
                        if ((float)Hn[(size_t)i * n_q + j] != (float)Hn[(size_t)j * n_q + i]) return false;      // not symmetric
                if (a <= b) { mblocks[n].push_back({n, a, b}); cost[n] += (size_t)len(a) * ld(b); }
            }
    }
    // modes to CTAs: largest first, to the least loaded CTA that still has a mode slot
    std::vector<int> order(n_phi);
    for (int n = 0; n < n_phi; ++n) order[n] = n;
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return cost[x] > cost[y]; });
    std::vector<size_t> load(G, 0);
    L.cta_nmodes.assign(G, 0); L.cta_modes.assign((size_t)G * RP_MAXM, -1);
    for (int n : order) {
        int best = -1;
        for (int g = 0; g < G; ++g) if (L.cta_nmodes[g] < RP_MAXM && (best < 0 || load[g] < load[best])) best = g;
        if (best < 0) return false;
        L.cta_modes[(size_t)best * RP_MAXM + L.cta_nmodes[best]++] = n; load[best] += cost[n];
    }
    // per CTA: pack the blocks, cut the items, write the tables
    L.cta_hoff.assign(G, 0); L.cta_hfloats.assign(G, 0); L.cta_cp.assign(G, 0); L.cta_rp.assign(G, 0);
    L.tab.assign((size_t)G * RP_CTA_STRIDE, 0);
    size_t least = (size_t)-1;
    for (int g = 0; g < G; ++g) {
        int *T = L.tab.data() + (size_t)g * RP_CTA_STRIDE;
        // a block with a != b may be stored either way round (it is its own mirror image): the ROW class pays the long join (one partial
        // per quad of columns, the column class one per chunk of rows), so the roles are dealt out evenly over the classes of the CTA
        std::vector<ReplBlock> blocks;
        std::vector<int> rowjoins(ncls, 0);
        for (int m = 0; m < L.cta_nmodes[g]; ++m)
            for (ReplBlock b : mblocks[L.cta_modes[(size_t)g * RP_MAXM + m]]) {
                if (b.a != b.b) {
                    if (rowjoins[b.b] < rowjoins[b.a]) std::swap(b.a, b.b);
                    rowjoins[b.a] += ld(b.b) / 4;
                }
                blocks.push_back(b);
            }
        int quads = 0;
        for (const ReplBlock &b : blocks) quads += ld(b.b) / 4;
        int nchunks = quads ? RP_THREADS / quads : 1;
        if (quads > RP_THREADS) return false;
        int rows_longest = 0;
        for (const ReplBlock &b : blocks) rows_longest = std::max(rows_longest, len(b.a));
        nchunks = std::max(1, std::min(nchunks, rows_longest));
        L.cta_hoff[g] = L.Hp.size();
        int *items = T + RP_HDR, *joins = T + RP_HDR + RP_THREADS * RP_ITEM;
        for (int t = 0; t < RP_THREADS; ++t) items[t * RP_ITEM + 5] = -1;
        int hoff = 0, cp = 0, rp = 0, t = 0;
        for (const ReplBlock &b : blocks) {
            const int la = len(b.a), lb = len(b.b), ldb = ld(b.b), nq4 = ldb / 4;
            const double *Hn = H + (size_t)b.n * n_q * n_q;
            for (int i = 0; i < la; ++i)
                for (int j = 0; j < ldb; ++j)
                    L.Hp.push_back(j < lb ? (float)Hn[(size_t)(class_start[b.a] + i) * n_q + class_start[b.b] + j] : 0.f);
            const bool rows = b.a != b.b;
            int slot = 0;
            while (L.cta_modes[(size_t)g * RP_MAXM + slot] != b.n) ++slot;
            const int rpitch = nq4 | 1;                                            // odd: thread k reads row k of rpart without bank conflicts
            const int RC = (la + nchunks - 1) / nchunks, nc = (la + RC - 1) / RC;
            L.rows_max = std::max(L.rows_max, RC);
            for (int j = 0; j < nc; ++j)
                for (int cq = 0; cq < nq4; ++cq, ++t) {
                    int *I = items + t * RP_ITEM;
                    const int r0 = j * RC, nr = std::min(RC, la - r0);
                    I[0] = hoff + r0 * ldb + 4 * cq; I[1] = ldb | (slot << 16); I[2] = class_start[b.a] + r0; I[3] = nr; I[4] = class_start[b.b] + 4 * cq;
                    I[5] = rows ? rp + r0 * rpitch + cq : -1; I[6] = rpitch; I[7] = cp + j * ldb + 4 * cq;
                }
            int *Jb = joins + (slot * RP_MAXCLS + b.b) * RP_JOIN;                  // the column class: column sums
            if (Jb[0]) return false;                                               // a class with two partner classes in one mode: not this kernel's case
            Jb[0] = 1; Jb[1] = cp; Jb[2] = nc; Jb[3] = ldb;
            if (rows) { int *Ja = joins + (slot * RP_MAXCLS + b.a) * RP_JOIN; if (Ja[0]) return false; Ja[0] = 2; Ja[1] = rp; Ja[2] = nq4; Ja[3] = rpitch; }
            hoff += la * ldb; cp += nc * ldb; if (rows) rp += la * rpitch;
        }
        if (t > RP_THREADS) return false;
        T[0] = (int)(L.cta_hoff[g] / 4); T[1] = hoff; T[2] = L.cta_nmodes[g]; T[3] = t;
        for (int m = 0; m < RP_MAXM; ++m) T[4 + m] = L.cta_modes[(size_t)g * RP_MAXM + m];
        L.cta_hfloats[g] = hoff; L.cta_cp[g] = cp; L.cta_rp[g] = rp;
        L.hfloats_max = std::max(L.hfloats_max, hoff); L.cp_max = std::max(L.cp_max, cp); L.rp_max = std::max(L.rp_max, rp);
        if (load[g] < least) { least = load[g]; L.out_cta = g; }
    }
    return (size_t)L.hfloats_max + L.cp_max + L.rp_max <= cap_floats;
}

}  // namespace modal_host
