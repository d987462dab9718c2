/* ewald_octplan.cpp -- host plan for the octant-form reciprocal kernel (ewald_recip_oct.cuh).
 *
 * From the G+ list of ewald_setup (Eq. 3's reciprocal sum) builds, for orthorhombic
 * cells, the non-negative octant n >= 0 with weights w(G_n) 2^nz, cut into items (column, n1 block),
 * and the per-CTA lane assignment that keeps every warp at one block length.  Long double where
 * values are computed (setup always in DP or better).
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
    const int nm0 = t->n_max[0], nm1 = t->n_max[1], nm2 = dim == 3 ? t->n_max[2] : 0;
    if (nm1 + nm2 + nm0 + 3 > 0xffff) return;
    const int nblk_max = std::max(1, (nm0 + 6) / 7);
    int npb = (nm0 + nblk_max - 1) / nblk_max;
    if (npb < 4) npb = 4;
    P.dim = dim;
    P.npb = npb;
    P.off[0] = 0;
    P.off[1] = nm0;
    P.off[2] = nm0 + nm1 + 1;
    P.rowlen = dim == 3 ? P.off[2] + nm2 + 1 : P.off[2];

    /* columns: (a, b, n1max_a, n1max_b); 3D: a = n2, b = n3; 2D: a, b = two n2 values (b = -1: none) */
    struct Col { int a, b, m; };
    std::vector<Col> cols;
    auto n1max_of = [&](int n2, int n3) {
        int m = -1;
        for (int n1 = 0; n1 <= nm0; n1++)
            if ((n1 == 0 && n2 == 0 && n3 == 0) || weight(n1, n2, n3) != 0.0) m = n1;
        return m;
    };
    if (dim == 3) {
        for (int n2 = 0; n2 <= nm1; n2++)
            for (int n3 = 0; n3 <= nm2; n3++) {
                const int m = n1max_of(n2, n3);
                if (m >= 0) cols.push_back({n2, n3, m});
            }
    } else {
        std::vector<std::pair<int, int>> v; /* (-n1max, n2) */
        for (int n2 = 0; n2 <= nm1; n2++) {
            const int m = n1max_of(n2, 0);
            if (m >= 0) v.push_back({-m, n2});
        }
        std::sort(v.begin(), v.end());
        for (size_t i = 0; i < v.size(); i += 2)
            cols.push_back({v[i].second, i + 1 < v.size() ? v[i + 1].second : -1, -v[i].first});
    }
    for (const Col &c : cols) {
        const int nblk = std::max(1, (c.m + npb - 1) / npb);
        for (int b = 0; b < nblk; b++) {
            const int start = b * npb, np = std::max(0, std::min(npb, c.m - start));
            P.offA.push_back(P.off[1] + c.a);
            P.offB.push_back(dim == 3 ? P.off[2] + c.b : P.off[1] + (c.b >= 0 ? c.b : c.a));
            P.offX.push_back(P.off[0] + start);
            P.np.push_back(np);
            P.c0.push_back(b == 0);
            P.col.push_back(c.a); P.col.push_back(c.b); P.col.push_back(start);
            for (int j = 0; j <= npb; j++) {
                const int n1 = j == 0 ? 0 : start + j;
                double wv[4] = {0, 0, 0, 0};
                if ((j == 0 && b == 0) || (j >= 1 && j <= np)) {
                    if (dim == 3) {
                        for (int cls = 0; cls < 4; cls++) wv[cls] = class_weight(n1, c.a, c.b, cls);
                    } else {
                        for (int cls = 0; cls < 2; cls++) {
                            wv[cls] = class_weight(n1, c.a, 0, cls);
                            wv[2 + cls] = c.b >= 0 ? class_weight(n1, c.b, 0, cls) : 0.0;
                        }
                    }
                }
                for (int cls = 0; cls < 4; cls++) P.wt.push_back(wv[cls]);
            }
        }
    }
    P.n_items = (int)P.np.size();
    P.valid = P.n_items > 0;
}

/* T_abc of the fixed charges per item entry, laid out like the kernel's accumulators. */
void fill_oct_ion(HostTables *t)
{
    OctPlan &P = t->oct;
    P.tion.clear();
    if (!P.valid || t->n_ion == 0) return;
    const int ne = 1 + 2 * P.npb, dim = t->dim;
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
        const int a = P.col[3 * it], b = P.col[3 * it + 1], start = P.col[3 * it + 2];
        for (int e = 0; e < ne; e++) {
            const int j = (e + 1) / 2, n1 = e == 0 ? 0 : start + j, which1 = e == 0 ? 0 : (e % 2 == 0);
            if (e == 0 && !P.c0[it]) continue;
            if (j > P.np[it]) continue;
            for (int k = 0; k < 4; k++) {
                real sum = 0;
                for (int i = 0; i < t->n_ion; i++) {
                    real pr;
                    if (dim == 3) pr = cs(i, 1, a, k >> 1) * cs(i, 2, b, k & 1);
                    else pr = k < 2 ? cs(i, 1, a, k & 1) : (b >= 0 ? cs(i, 1, b, k & 1) : 0);
                    sum += (real)t->ion_q[i] * pr * cs(i, 0, n1, which1);
                }
                P.tion[((size_t)it * ne + e) * 4 + k] = (double)sum;
            }
        }
    }
}

void make_oct_launch(const OctPlan &P, int wc, int max_warps, OctLaunch *L)
{
    struct Key { int len, wl, item; };
    std::vector<Key> v;
    v.reserve((size_t)wc * P.n_items);
    for (int wl = 0; wl < wc; wl++)
        for (int it = 0; it < P.n_items; it++) v.push_back({2 * P.np[it] + P.c0[it], wl, it});
    std::sort(v.begin(), v.end(), [](const Key &x, const Key &y) {
        if (x.len != y.len) return x.len > y.len;
        if (x.wl != y.wl) return x.wl < y.wl;
        return x.item < y.item;
    });
    /* the sorted list is cut into n_slabs CTAs of n_warps warps each (one CTA when it fits) */
    const int total_warps = (int)((v.size() + 31) / 32);
    const int n_slabs = (total_warps + max_warps - 1) / max_warps;
    const int per_cta = (total_warps + n_slabs - 1) / n_slabs;
    const int n_warps = per_cta * n_slabs; /* padded: trailing warps hold dummy items only */
    L->wc = wc;
    L->n_warps = per_cta;
    L->n_slabs = n_slabs;
    L->lane.assign((size_t)n_warps * 32 * 4, 0);
    L->variant.assign(n_warps, 0);
    L->cost = 0;
    /* padding lanes repeat the list's last entry with item = a zero-weight dummy: item index n_items */
    /* rank = position of a lane among the lanes of its walker inside its CTA: the kernel adds a walker's
     * lane sums in rank order, so the result does not depend on where in the batch the walker sits */
    std::vector<int> next_rank((size_t)wc, 0);
    L->rank_stride = 1;
    for (int wp = 0; wp < n_warps; wp++) {
        if (wp % per_cta == 0) std::fill(next_rank.begin(), next_rank.end(), 0);
        int np = 0, c0 = 0;
        for (int l = 0; l < 32; l++) {
            const size_t i = (size_t)wp * 32 + l;
            int *o = &L->lane[i * 4];
            if (i < v.size()) {
                const Key &k = v[i];
                const int rank = next_rank[k.wl]++;
                if (rank + 1 > L->rank_stride) L->rank_stride = rank + 1;
                o[0] = k.wl | (rank << 8); o[1] = k.item;
                o[2] = P.offA[k.item] | (P.offB[k.item] << 16);
                o[3] = P.offX[k.item];
                np = std::max(np, P.np[k.item]);
                c0 = std::max(c0, P.c0[k.item]);
            } else {
                o[0] = 0 | (0xffffff << 8); o[1] = P.n_items; /* dummy item: all weights zero, no rank */
                o[2] = P.offA[0] | (P.offB[0] << 16);
                o[3] = P.offX[0];
            }
        }
        L->variant[wp] = np | (c0 << 8);
        if ((size_t)wp * 32 < v.size()) L->cost += 32.0 * (4.0 * (2 * np + c0) + (P.dim == 3 ? 4.0 : 0.0));
    }
}

} // namespace ewald
