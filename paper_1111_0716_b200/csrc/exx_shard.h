// exx_shard.h — the batch list of the fused loop nest and its assignment to shards.
// Host-only, no CUDA: used by the pair loop of exx_fused.cu and by exx_shard_plan (callable without a GPU).
// Product code: shares nothing with oracle/.
//
// The loop nest (k and q loops, then the band loops, innermost blocked) is cut into batches: one
// (a-tile at k-point k) x (b-tile at k-point q) block of at most tile x tile band pairs.  Every batch is independent of every
// other one except for the accumulators it adds to, and S7 (forward transform + gather) is linear, so a shard may run any
// subset of the batches, finish S7 on its partial accumulators, and the shards' outputs are summed once (one all-reduce of
// the sphere coefficients, 40 MB at C4a) — no accumulator box ever crosses the link.
#pragma once
#include <stdint.h>

#include <algorithm>
#include <vector>

namespace exx {

struct PairBlock {
    int k, q;          // k-points of the a-bands and the b-bands
    int a0, ta;        // a-bands a0 .. a0+ta-1
    int b0, tb;        // positions b0 .. b0+tb-1 of the b-band list of (q, mode)
    int npairs;        // pair densities transformed (passes A, B)
    int units_a;       // pass-C accumulations into the a-bands
    int units_b;       // pass-C accumulations into the b-bands (pair symmetry only)
    int shard;
    int64_t cost() const { return 2 * (int64_t)npairs + units_a + units_b; }  // pass executions
};

// b-bands of k-point q: with the pair symmetry every band (an empty band still receives), else the bands with f != 0
inline void b_list(int nb, const double* occ, int q, bool sym, std::vector<int>& out) {
    out.clear();
    for (int m = 0; m < nb; m++)
        if (sym || occ[q * nb + m] != 0.0) out.push_back(m);
}

// is the pair (a at k, b at q) transformed?  plain: iff f_b != 0; symmetry: each unordered pair once, iff either side is occupied
inline bool pair_evaluated(bool sym, int k, int q, int a, int b, double fa, double fb) {
    return sym ? ((fa != 0.0 || fb != 0.0) && (k < q || a <= b)) : (fb != 0.0);
}

// All non-empty batches in loop order, each assigned to a shard: longest-processing-time first (batches sorted by cost,
// ties in loop order, each to the least loaded shard, ties to the lowest rank) — deterministic, the same on every rank.
// na: number of a-bands per k-point (default nb; exx_apply_to with a block of na trial vectors: a = 0 .. na-1, needs !sym)
inline void plan_blocks(int nk, int nb, const double* occ, bool sym, int ta_max, int tb_max, int nshards, std::vector<PairBlock>& out, int na = -1) {
    out.clear();
    if (na < 0) na = nb;
    std::vector<int> blist;
    for (int k = 0; k < nk; k++)
        for (int q = sym ? k : 0; q < nk; q++) {
            b_list(nb, occ, q, sym, blist);
            for (int a0 = 0; a0 < na; a0 += ta_max)
                for (size_t b0 = (sym && k == q) ? (size_t)a0 : 0; b0 < blist.size(); b0 += tb_max) {
                    PairBlock p;
                    p.k = k, p.q = q, p.a0 = a0, p.b0 = (int)b0;
                    p.ta = std::min(ta_max, na - a0);
                    p.tb = (int)std::min<size_t>(tb_max, blist.size() - b0);
                    p.npairs = p.units_a = p.units_b = 0;
                    p.shard = 0;
                    for (int i = 0; i < p.ta; i++)
                        for (int j = 0; j < p.tb; j++) {
                            const int a = a0 + i, b = blist[b0 + j];
                            const double fa = a < nb ? occ[k * nb + a] : 0.0, fb = occ[q * nb + b];  // (fa is used with sym only)
                            if (!pair_evaluated(sym, k, q, a, b, fa, fb)) continue;
                            p.npairs++;
                            if (fb != 0.0) p.units_a++;
                            if (sym && fa != 0.0 && !(k == q && a == b)) p.units_b++;
                        }
                    if (p.npairs) out.push_back(p);
                }
        }
    if (nshards <= 1) return;
    std::vector<int> order(out.size());
    for (size_t i = 0; i < order.size(); i++) order[i] = (int)i;
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return out[x].cost() > out[y].cost(); });
    std::vector<int64_t> load(nshards, 0);
    for (int i : order) {
        int best = 0;
        for (int s = 1; s < nshards; s++)
            if (load[s] < load[best]) best = s;
        out[i].shard = best;
        load[best] += out[i].cost();
    }
}

}  // namespace exx
