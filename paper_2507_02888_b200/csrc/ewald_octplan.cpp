/* ewald_octplan.cpp -- host plan for the octant-form reciprocal kernel (ewald_recip_oct.cuh).
 *
 * From the G+ list of ewald_setup (Eq. 3's reciprocal sum) builds the non-negative octant
 * n >= 0 with the class weights of every octant point, cut into items (column(s), n1 block), and the per-CTA
 * lane assignment: warps of one block length, dealt to the four sub-partitions of an SM so that they carry
 * equal FP64 work.  Long double where values are computed (setup always in DP or better).
 */
#include <algorithm>
#include <cmath>
#include <map>
#include <tuple>

#include "ewald_internal.h"

namespace ewald {

typedef long double real;
static const real kPi = 3.141592653589793238462643383279502884L;

void build_oct_plan(HostTables *t)
{
    OctPlan &P = t->oct;
    P = OctPlan();
    /* Any cell: G.r = 2 pi n.s in fractional coordinates, so the eight real sums T_abc(n), n >= 0, give
     * rho(+-n1, +-n2, +-n3) for every sign choice.  Only the weights depend on the signs when the reciprocal
     * axes are not orthogonal: rho(-G) = conj rho(G) leaves four classes (p, q) = (s1 s2, s1 s3), each with
     * its own weight W_pq(n) = 2^nz/4 w(n1, p n2, q n3) (2^nz/8 per sign choice corrects for the choices that
     * coincide when some n_k = 0; times 2 for G and -G).  2D: two classes p, W_p = 2^nz/2 w(n1, p n2). */
    const int dim = t->dim;
    const size_t ngp = t->g_w2.size();
    std::map<std::tuple<int, int, int>, double> w; /* full-sphere weight w(G) = w2 / 2, keyed by the half-set member */
    for (size_t g = 0; g < ngp; g++)
        w[std::make_tuple(t->g_n[3 * g], t->g_n[3 * g + 1], t->g_n[3 * g + 2])] = 0.5 * t->g_w2[g];
    auto w_of = [&](int n1, int n2, int n3) -> double { /* w(G) for any signs, 0 outside the sphere */
        if (n1 < 0 || (n1 == 0 && (n2 < 0 || (n2 == 0 && n3 < 0)))) { n1 = -n1; n2 = -n2; n3 = -n3; }
        auto it = w.find(std::make_tuple(n1, n2, n3));
        return it == w.end() ? 0.0 : it->second;
    };
    /* class weights of the octant point n >= 0: 3D (++, +-, -+, --) in (p, q); 2D (+, -) in p */
    auto class_weight = [&](int n1, int n2, int n3, int cls) -> double {
        const int nz = (n1 != 0) + (n2 != 0) + (n3 != 0);
        if (dim == 3) {
            const int p = (cls & 2) ? -1 : 1, q = (cls & 1) ? -1 : 1;
            return w_of(n1, p * n2, q * n3) * (double)(1 << nz) / 4.0;
        }
        return w_of(n1, (cls & 1) ? -n2 : n2, 0) * (double)(1 << nz) / 2.0;
    };
    auto weight = [&](int n1, int n2, int n3) -> double { /* sum over the classes: non-zero iff the point is used */
        double sum = 0;
        for (int cls = 0; cls < (dim == 3 ? 4 : 2); cls++) sum += class_weight(n1, n2, n3, cls);
        return sum;
    };
    /* A half column is a column with one phase only: (n2, 0) [axis 1], (0, n3) [axis 2]; in 2D every column.
     * Its two sign classes s = +-: the class weights of the point summed over the sign that does not matter. */
    auto half_weight = [&](int n1, int axis, int n, int s) -> double {
        if (dim == 2) return class_weight(n1, n, 0, s);
        if (axis == 1) return class_weight(n1, n, 0, 2 * s) + class_weight(n1, n, 0, 2 * s + 1);
        return class_weight(n1, 0, n, s) + class_weight(n1, 0, n, 2 + s);
    };
    const int nm0 = t->n_max[0], nm1 = t->n_max[1], nm2 = dim == 3 ? t->n_max[2] : 0;
    if (nm1 + nm2 + nm0 + 3 > 0xffff) return;
    const int nblk_max = std::max(1, (nm0 + 6) / 7);
    int npb = (nm0 + nblk_max - 1) / nblk_max;
    if (npb < 4) npb = 4;
    P.dim = dim;
    P.npb = npb;
    /* table row of one (walker, particle): X1[0..nm0] (carries q), X2[0..nm1], X3[0..nm2] as (cos, sin) pairs */
    P.off[0] = 0;
    P.off[1] = nm0 + 1;
    P.off[2] = nm0 + nm1 + 2;
    P.rowlen = dim == 3 ? P.off[2] + nm2 + 1 : P.off[2];
    P.rowlen |= 1; /* odd number of 16-byte pairs: 32 lanes that write (or read) the same entry of 32 consecutive rows hit 32 different bank groups */

    auto n1max_of = [&](int n2, int n3) {
        int m = -1;
        for (int n1 = 0; n1 <= nm0; n1++)
            if ((n1 == 0 && n2 == 0 && n3 == 0) || weight(n1, n2, n3) != 0.0) m = n1;
        return m;
    };
    /* columns: FULL (n2 > 0 and n3 > 0: four products X2 (x) X3) and half columns, paired two to an item */
    struct Col { int kind, aa, an, ba, bn, m; }; /* kind, half A (axis, n), half B (axis, n; axis -1: none), n1max */
    struct Half { int m, axis, n; };
    std::vector<Col> cols;
    std::vector<Half> halves;
    if (dim == 3) {
        for (int n2 = 0; n2 <= nm1; n2++)
            for (int n3 = 0; n3 <= nm2; n3++) {
                const int m = n1max_of(n2, n3);
                if (m < 0) continue;
                if (n2 > 0 && n3 > 0) cols.push_back({OCT_FULL, 1, n2, 2, n3, m});
                else halves.push_back({m, n3 > 0 ? 2 : 1, n3 > 0 ? n3 : n2});
            }
    } else {
        for (int n2 = 0; n2 <= nm1; n2++) {
            const int m = n1max_of(n2, 0);
            if (m >= 0) halves.push_back({m, 1, n2});
        }
    }
    std::sort(halves.begin(), halves.end(), [](const Half &x, const Half &y) {
        if (x.m != y.m) return x.m > y.m;
        if (x.axis != y.axis) return x.axis < y.axis;
        return x.n < y.n;
    });
    for (size_t i = 0; i < halves.size(); i += 2) {
        const bool two = i + 1 < halves.size();
        cols.push_back({OCT_PAIR, halves[i].axis, halves[i].n, two ? halves[i + 1].axis : -1, two ? halves[i + 1].n : 0,
                        halves[i].m});
    }
    auto half_off = [&](int axis, int n) { return P.off[axis] + n; };
    for (const Col &c : cols) {
        const int nblk = std::max(1, (c.m + npb - 1) / npb);
        for (int b = 0; b < nblk; b++) {
            const int start = b * npb, np = std::max(0, std::min(npb, c.m - start));
            P.kind.push_back(c.kind);
            P.offA.push_back(half_off(c.aa, c.an));
            P.offB.push_back(c.ba >= 0 ? half_off(c.ba, c.bn) : half_off(c.aa, c.an));
            P.offX.push_back(P.off[0] + start); /* pairs j = 1..np at offX + j; block 0 also reads offX + 0 = (q, 0) */
            P.np.push_back(np);
            P.c0.push_back(b == 0);
            P.col.push_back(c.aa); P.col.push_back(c.an); P.col.push_back(c.ba); P.col.push_back(c.bn); P.col.push_back(start);
            for (int j = 0; j <= npb; j++) {
                const int n1 = j == 0 ? 0 : start + j;
                double wv[4] = {0, 0, 0, 0};
                if ((j == 0 && b == 0) || (j >= 1 && j <= np)) {
                    if (c.kind == OCT_FULL) {
                        for (int cls = 0; cls < 4; cls++) wv[cls] = class_weight(n1, c.an, c.bn, cls);
                    } else {
                        for (int s = 0; s < 2; s++) {
                            wv[s] = half_weight(n1, c.aa, c.an, s);
                            wv[2 + s] = c.ba >= 0 ? half_weight(n1, c.ba, c.bn, s) : 0.0;
                        }
                    }
                }
                for (int cls = 0; cls < 4; cls++) P.wt.push_back(wv[cls]);
            }
        }
    }
    P.n_items = (int)P.np.size();
    P.valid = P.n_items > 0;

    /* ---- the tensor-core (DMMA) form of the same sums: groups of 8 columns, M-tiles of 4 n1 values ---- */
    MmaPlan &M = t->mma;
    M = MmaPlan();
    M.dim = dim; M.rowlen = P.rowlen;
    for (int k = 0; k < 3; k++) M.off[k] = P.off[k];
    struct MCol { int ax0, n0, ax1, n1, m; };  /* FULL: (1, n2, 2, n3); HALF: (axis, n, -1, 0) */
    auto tiles_of = [](int m) { return m / 4 + 1; };
    /* two columns that share a quarter-warp read two 64-byte chunks (entry x 4 particles) of one operand in one
     * LDS.128: without bank conflict when the entries are equal or differ in parity */
    auto compatible = [&](const MCol &x, const MCol &y) {
        auto ok = [&](int ax, int a, int bx, int b) {
            const int ea = P.off[ax] + a, eb = P.off[bx] + b; /* entries within a table row */
            return ea == eb || ((ea + eb) & 1) != 0;
        };
        return ok(x.ax0, x.n0, y.ax0, y.n0) && (x.ax1 < 0 || ok(x.ax1, x.n1, y.ax1, y.n1));
    };
    auto make_groups = [&](std::vector<MCol> v) {
        std::stable_sort(v.begin(), v.end(), [&](const MCol &x, const MCol &y) { return tiles_of(x.m) > tiles_of(y.m); });
        std::vector<std::vector<MCol>> groups;
        for (size_t i = 0; i < v.size(); i += 8) {
            std::vector<MCol> g(v.begin() + i, v.begin() + std::min(v.size(), i + 8));
            /* greedy pairing for the quarter-warps */
            std::vector<MCol> out;
            std::vector<bool> used(g.size(), false);
            for (size_t a = 0; a < g.size(); a++) {
                if (used[a]) continue;
                used[a] = true;
                out.push_back(g[a]);
                size_t best = g.size();
                for (size_t b = a + 1; b < g.size(); b++)
                    if (!used[b] && compatible(g[a], g[b])) { best = b; break; }
                if (best == g.size())
                    for (size_t b = a + 1; b < g.size(); b++)
                        if (!used[b]) { best = b; break; }
                if (best < g.size()) { used[best] = true; out.push_back(g[best]); }
            }
            groups.push_back(out);
        }
        return groups;
    };
    std::vector<MCol> fullc, halfc;
    for (const Col &c : cols)
        if (c.kind == OCT_FULL) fullc.push_back({1, c.an, 2, c.bn, c.m});
    for (const Half &h : halves) halfc.push_back({h.axis, h.n, -1, 0, h.m});
    const auto fgroups = make_groups(fullc), hgroups = make_groups(halfc);
    auto group_tiles = [&](const std::vector<MCol> &g) { int tl = 1; for (const MCol &c : g) tl = std::max(tl, tiles_of(c.m)); return tl; };
    auto push_slot = [&](int kind, const std::vector<MCol> *ga, const std::vector<MCol> *gb, int t0, int nt) {
        MmaSlot S;
        S.kind = kind; S.t0 = t0; S.nt = nt;
        for (int c = 0; c < 8; c++) {
            S.ax[0][c] = S.ax[1][c] = -1; S.n[0][c] = S.n[1][c] = 0;
            if (kind == OCT_FULL) {
                if (c < (int)ga->size()) { S.ax[0][c] = 1; S.n[0][c] = (*ga)[c].n0; S.ax[1][c] = 2; S.n[1][c] = (*ga)[c].n1; }
            } else {
                if (c < (int)ga->size()) { S.ax[0][c] = (*ga)[c].ax0; S.n[0][c] = (*ga)[c].n0; }
                if (gb && c < (int)gb->size()) { S.ax[1][c] = (*gb)[c].ax0; S.n[1][c] = (*gb)[c].n0; }
            }
        }
        for (int tile = 0; tile < 2; tile++)
            for (int l = 0; l < 4; l++) {
                const int n1 = 4 * (t0 + tile) + l;
                for (int c = 0; c < 8; c++)
                    for (int cls = 0; cls < 4; cls++) {
                        double wv = 0;
                        if (tile < nt && n1 <= nm0) {
                            if (kind == OCT_FULL) { if (S.ax[0][c] >= 0) wv = class_weight(n1, S.n[0][c], S.n[1][c], cls); }
                            else if (S.ax[cls >> 1][c] >= 0) wv = half_weight(n1, S.ax[cls >> 1][c], S.n[cls >> 1][c], cls & 1);
                        }
                        M.wt.push_back(wv);
                    }
            }
        M.slots.push_back(S);
        M.dmma_per_quad += 4.0 * nt;
    };
    for (const auto &g : fgroups)
        for (int t0 = 0; t0 < group_tiles(g); t0 += 2) push_slot(OCT_FULL, &g, nullptr, t0, std::min(2, group_tiles(g) - t0));
    for (size_t i = 0; i < hgroups.size(); i += 2) {
        const std::vector<MCol> *ga = &hgroups[i], *gb = i + 1 < hgroups.size() ? &hgroups[i + 1] : nullptr;
        const int tl = std::max(group_tiles(*ga), gb ? group_tiles(*gb) : 1);
        for (int t0 = 0; t0 < tl; t0 += 2) push_slot(OCT_PAIR, ga, gb, t0, std::min(2, tl - t0));
    }
    M.valid = !M.slots.empty() && dim >= 2;
}

/* T_abc of the fixed charges per item entry, laid out like the kernel's accumulators: entry e = 0 is n1 = 0
 * (cos only), e = 2j - 1 / 2j the cos / sin of n1 = start + j; products k as in the kernel (FULL: c2c3, c2s3,
 * s2c3, s2s3; PAIR: cos, sin of half A, cos, sin of half B). */
void fill_oct_ion(HostTables *t)
{
    OctPlan &P = t->oct;
    P.tion.clear();
    if (!P.valid || t->n_ion == 0) return;
    const int ne = 1 + 2 * P.npb;
    P.tion.assign((size_t)P.n_items * ne * 4, 0.0);
    std::vector<real> s((size_t)3 * t->n_ion);
    for (int i = 0; i < t->n_ion; i++)
        for (int k = 0; k < 3; k++) {
            real v = 0;
            for (int x = 0; x < 3; x++) v += (real)t->ion_pos[3 * i + x] * (real)t->binv[3 * k + x];
            s[3 * i + k] = v - nearbyintl(v);
        }
    auto cs = [&](int i, int k, int n, int which) -> real {
        real ph = n * s[3 * i + k];
        ph -= nearbyintl(ph);
        return which ? sinl(2 * kPi * ph) : cosl(2 * kPi * ph);
    };
    for (int it = 0; it < P.n_items; it++) {
        const int *c = &P.col[5 * it];
        const int aa = c[0], an = c[1], ba = c[2], bn = c[3], start = c[4];
        for (int e = 0; e < ne; e++) {
            const int j = (e + 1) / 2, n1 = e == 0 ? 0 : start + j, which1 = e == 0 ? 0 : (e % 2 == 0);
            if (e == 0 && !P.c0[it]) continue;
            if (j > P.np[it]) continue;
            for (int k = 0; k < 4; k++) {
                real sum = 0;
                for (int i = 0; i < t->n_ion; i++) {
                    real pr;
                    if (P.kind[it] == OCT_FULL) pr = cs(i, aa, an, k >> 1) * cs(i, ba, bn, k & 1);
                    else pr = k < 2 ? cs(i, aa, an, k & 1) : (ba >= 0 ? cs(i, ba, bn, k & 1) : 0);
                    sum += (real)t->ion_q[i] * pr * cs(i, 0, n1, which1);
                }
                P.tion[((size_t)it * ne + e) * 4 + k] = (double)sum;
            }
        }
    }
}

/* Lane assignment of the CTAs of one group of `wc` walkers.  The (walker, item) lanes are sorted by kind and
 * block length and cut into warps (a warp never mixes kinds and runs the block length of its longest lane).
 * The warps are then dealt to n_slabs CTAs x 4 sub-partitions, longest first to the least loaded bin (warp w of
 * a CTA runs on sub-partition w mod 4): the FMA phase of a CTA lasts as long as its busiest sub-partition. */
void make_oct_launch(const OctPlan &P, int wc, int max_warps, OctLaunch *L)
{
    struct Key { int kind, len, wl, item; };
    std::vector<Key> v;
    v.reserve((size_t)wc * P.n_items);
    for (int wl = 0; wl < wc; wl++)
        for (int it = 0; it < P.n_items; it++) v.push_back({P.kind[it], 2 * P.np[it] + P.c0[it], wl, it});
    std::sort(v.begin(), v.end(), [](const Key &x, const Key &y) {
        if (x.kind != y.kind) return x.kind < y.kind;
        if (x.len != y.len) return x.len > y.len;
        if (x.wl != y.wl) return x.wl < y.wl;
        return x.item < y.item;
    });
    struct Warp { size_t first, count; int kind, np, c0; double cost; };
    std::vector<Warp> warps;
    for (size_t i = 0; i < v.size();) {
        size_t j = i;
        int np = 0, c0 = 0;
        while (j < v.size() && j - i < 32 && v[j].kind == v[i].kind) {
            np = std::max(np, P.np[v[j].item]);
            c0 = std::max(c0, P.c0[v[j].item]);
            j++;
        }
        /* FP64 operations per particle of one lane: the tile's FMAs and the products */
        warps.push_back({i, j - i, v[i].kind, np, c0, 4.0 * (2 * np + c0) + (v[i].kind == OCT_FULL ? 4.0 : 0.0)});
        i = j;
    }
    max_warps = std::max(4, max_warps);
    const int total = (int)warps.size();
    const int n_slabs = std::max(1, (total + max_warps - 1) / max_warps);
    const int n_bins = 4 * n_slabs;
    auto bin_cap = [&](int b) { return (max_warps - (b & 3) + 3) / 4; }; /* warps w = b mod 4, + 4, ... below max_warps */
    std::vector<std::vector<int>> bins(n_bins);
    std::vector<double> load(n_bins, 0.0);
    std::vector<int> order(total);
    for (int i = 0; i < total; i++) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return warps[a].cost > warps[b].cost; });
    for (int wi : order) {
        int best = -1;
        for (int b = 0; b < n_bins; b++)
            if ((int)bins[b].size() < bin_cap(b) && (best < 0 || load[b] < load[best])) best = b;
        bins[best].push_back(wi);
        load[best] += warps[wi].cost;
    }
    int per_cta = 4;
    for (int b = 0; b < n_bins; b++)
        if (!bins[b].empty()) per_cta = std::max(per_cta, 4 * ((int)bins[b].size() - 1) + (b & 3) + 1);
    L->wc = wc;
    L->n_warps = per_cta;
    L->n_slabs = n_slabs;
    L->lane.assign((size_t)n_slabs * per_cta * 32 * 4, 0);
    L->variant.assign((size_t)n_slabs * per_cta, OCT_EMPTY << 16);
    L->cost = 32.0 * 4.0 * n_slabs * *std::max_element(load.begin(), load.end());
    L->fma_ops = 0;
    /* rank = position of the item in the sorted item list (the same for every walker): the kernel adds a
     * walker's lane sums in rank order, so the result does not depend on where in the batch the walker sits */
    std::vector<int> item_rank((size_t)P.n_items, 0);
    {
        int r = 0;
        for (const Key &k : v)
            if (k.wl == 0) item_rank[k.item] = r++;
    }
    L->rank_stride = P.n_items;
    for (int s = 0; s < n_slabs; s++) {
        for (int wp = 0; wp < per_cta; wp++) {
            const std::vector<int> &bin = bins[4 * s + (wp & 3)];
            const int slot = wp >> 2;
            const Warp *W = slot < (int)bin.size() ? &warps[bin[slot]] : nullptr;
            if (W) {
                L->variant[(size_t)s * per_cta + wp] = W->np | (W->c0 << 8) | (W->kind << 16);
                L->fma_ops += 32.0 * W->cost;
            }
            for (int l = 0; l < 32; l++) {
                int *o = &L->lane[(((size_t)s * per_cta + wp) * 32 + l) * 4];
                if (W && (size_t)l < W->count) {
                    const Key &k = v[W->first + l];
                    const int rank = item_rank[k.item];
                    o[0] = k.wl | (rank << 8); o[1] = k.item;
                    o[2] = P.offA[k.item] | (P.offB[k.item] << 16);
                    o[3] = P.offX[k.item];
                } else { /* dummy item (index n_items): all weights zero, no rank */
                    o[0] = 0 | (0xffffff << 8); o[1] = P.n_items;
                    o[2] = P.offA[0] | (P.offB[0] << 16);
                    o[3] = P.offX[0];
                }
            }
        }
    }
}

} // namespace ewald

namespace ewald {

/* Fixed-charge sums laid out like the DMMA accumulators: [slot][tile][X1 double d][column][product]. */
void fill_mma_ion(HostTables *t)
{
    MmaPlan &M = t->mma;
    M.tion.clear();
    if (!M.valid || t->n_ion == 0) return;
    M.tion.assign(M.slots.size() * 2 * 8 * 8 * 4, 0.0);
    std::vector<real> s((size_t)3 * t->n_ion);
    for (int i = 0; i < t->n_ion; i++)
        for (int k = 0; k < 3; k++) {
            real v = 0;
            for (int x = 0; x < 3; x++) v += (real)t->ion_pos[3 * i + x] * (real)t->binv[3 * k + x];
            s[3 * i + k] = v - nearbyintl(v);
        }
    auto cs = [&](int i, int k, int n, int which) -> real {
        real ph = n * s[3 * i + k];
        ph -= nearbyintl(ph);
        return which ? sinl(2 * kPi * ph) : cosl(2 * kPi * ph);
    };
    for (size_t si = 0; si < M.slots.size(); si++) {
        const MmaSlot &S = M.slots[si];
        for (int tile = 0; tile < S.nt; tile++)
            for (int d = 0; d < 8; d++) {
                const int idx = 8 * (S.t0 + tile) + d, n1 = idx >> 1, which1 = idx & 1;
                if (n1 > t->n_max[0]) continue;
                for (int c = 0; c < 8; c++)
                    for (int k = 0; k < 4; k++) {
                        real sum = 0;
                        for (int i = 0; i < t->n_ion; i++) {
                            real pr = 0;
                            if (S.kind == OCT_FULL) {
                                if (S.ax[0][c] >= 0) pr = cs(i, 1, S.n[0][c], k >> 1) * cs(i, 2, S.n[1][c], k & 1);
                            } else if (S.ax[k >> 1][c] >= 0) {
                                pr = cs(i, S.ax[k >> 1][c], S.n[k >> 1][c], k & 1);
                            }
                            sum += (real)t->ion_q[i] * pr * cs(i, 0, n1, which1);
                        }
                        M.tion[(((si * 2 + tile) * 8 + d) * 8 + c) * 4 + k] = (double)sum;
                    }
            }
    }
}

/* Deals the slots of one walker to wpw warps: longest first to the least loaded warp that still has room and
 * whose slots start at the same M-tile (the warp loads the X1 operand of a quad once for all its slots). */
void make_mma_launch(const MmaPlan &M, int wpw, MmaLaunch *L)
{
    L->wpw = wpw;
    L->valid = false;
    L->lane.assign((size_t)wpw * MMA_SMAX * 32 * 2, 0);
    L->meta.assign((size_t)wpw * MMA_SMAX * 4, 0);
    for (int w = 0; w < wpw; w++)
        for (int s = 0; s < MMA_SMAX; s++) L->meta[((size_t)w * MMA_SMAX + s) * 4] = OCT_EMPTY;
    /* classes of slots by first M-tile: the fewest warps each class needs, spare warps to the class with the most
     * work per warp; inside a class longest slot first to the least loaded warp */
    std::map<int, std::vector<int>> classes;
    for (size_t i = 0; i < M.slots.size(); i++) classes[M.slots[i].t0].push_back((int)i);
    std::map<int, int> n_w;
    std::map<int, double> work;
    int used = 0;
    for (auto &kv : classes) {
        n_w[kv.first] = ((int)kv.second.size() + MMA_SMAX - 1) / MMA_SMAX;
        used += n_w[kv.first];
        double wk = 0;
        for (int si : kv.second) wk += 4.0 * M.slots[si].nt;
        work[kv.first] = wk;
    }
    if (used > wpw) return; /* does not fit */
    for (; used < wpw; used++) {
        int best = -1;
        for (auto &kv : classes)
            if (n_w[kv.first] < (int)kv.second.size() && (best < 0 || work[kv.first] / n_w[kv.first] > work[best] / n_w[best]))
                best = kv.first;
        if (best < 0) break;
        n_w[best]++;
    }
    /* a piece = (slot, mask of its tiles): whole slots first, two-tile slots may be split to even the loads */
    struct Piece { int slot, mask; };
    std::vector<std::vector<Piece>> bins(wpw);
    std::vector<double> load(wpw, 0.0);
    std::vector<int> win(wpw, 0); /* first M-tile of the warp's two-tile window */
    int w_first = 0;
    for (auto &kv : classes) {
        std::vector<int> order(kv.second);
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return M.slots[a].nt > M.slots[b].nt; });
        const int w_end = w_first + n_w[kv.first];
        for (int w = w_first; w < w_end; w++) win[w] = kv.first;
        for (int si : order) {
            int best = -1;
            for (int w = w_first; w < w_end; w++)
                if ((int)bins[w].size() < MMA_SMAX && (best < 0 || load[w] < load[best])) best = w;
            if (best < 0) return;
            bins[best].push_back({si, M.slots[si].nt > 1 ? 3 : 1});
            load[best] += 4.0 * M.slots[si].nt;
        }
        /* the busiest warp of the class hands one tile of a two-tile slot to the idlest one while that helps */
        for (int guard = 0; guard < 64; guard++) {
            int hi = w_first, lo = w_first;
            for (int w = w_first; w < w_end; w++) {
                if (load[w] > load[hi]) hi = w;
                if (load[w] < load[lo]) lo = w;
            }
            if (load[hi] - load[lo] < 8.0 || (int)bins[lo].size() >= MMA_SMAX) break;
            size_t k = 0;
            while (k < bins[hi].size() && bins[hi][k].mask != 3) k++;
            if (k == bins[hi].size()) break;
            bins[hi][k].mask = 1;
            bins[lo].push_back({bins[hi][k].slot, 2});
            load[hi] -= 4.0; load[lo] += 4.0;
        }
        w_first = w_end;
    }
    /* heaviest warps first, so that warp w mod 4 (the sub-partition) sees every weight class in turn */
    {
        std::vector<int> perm(wpw);
        for (int w = 0; w < wpw; w++) perm[w] = w;
        std::stable_sort(perm.begin(), perm.end(), [&](int a, int b) { return load[a] > load[b]; });
        std::vector<std::vector<Piece>> b2(wpw);
        std::vector<double> l2(wpw);
        std::vector<int> w2(wpw);
        for (int w = 0; w < wpw; w++) { b2[w] = bins[perm[w]]; l2[w] = load[perm[w]]; w2[w] = win[perm[w]]; }
        bins.swap(b2); load.swap(l2); win.swap(w2);
    }
    L->max_dmma = 0;
    for (int w = 0; w < wpw; w++) {
        L->max_dmma = std::max(L->max_dmma, load[w]);
        for (size_t s = 0; s < bins[w].size(); s++) {
            const int si = bins[w][s].slot;
            const MmaSlot &S = M.slots[si];
            int *meta = &L->meta[((size_t)w * MMA_SMAX + s) * 4];
            /* kind, the warp's window, tile mask within the window, slot | first tile of the slot << 16 */
            meta[0] = S.kind; meta[1] = win[w]; meta[2] = bins[w][s].mask << (S.t0 - win[w]); meta[3] = si | (S.t0 << 16);
            for (int lane = 0; lane < 32; lane++) {
                const int kk = lane & 3, c = lane >> 2;
                int *o = &L->lane[(((size_t)w * MMA_SMAX + s) * 32 + lane) * 2];
                for (int h = 0; h < 2; h++) {
                    const int ax = S.ax[h][c] >= 0 ? S.ax[h][c] : 1, n = S.ax[h][c] >= 0 ? S.n[h][c] : 0;
                    o[h] = (M.off[ax] + n) * 4 + kk;
                }
            }
        }
    }
    L->valid = true;
}

} // namespace ewald
