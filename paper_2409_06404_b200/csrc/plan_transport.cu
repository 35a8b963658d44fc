// plan_transport.cu -- host code: the tile schedule and the schedule-ordered tables of
// transport_tiled.cu (see the header comment there and TransportPlan in crf_internal.h).
#include <cmath>
#include <cstdint>
#include <random>

#include "fastmath.cuh"
#include "host_plan.h"

namespace {

struct Tile {
    int jb, kb;
};

// Rounds of at most W off-diagonal tiles whose species blocks are pairwise disjoint.  Greedy: each round
// takes, among the tiles disjoint from those already chosen, the one whose blocks still have the most
// tiles left (ties broken by a seeded shuffle); several seeds, fewest rounds wins.
std::vector<std::vector<Tile>> schedule_offdiag(int nb, int W)
{
    std::vector<std::vector<Tile>> best;
    const int ntiles = nb * (nb - 1) / 2;
    if (ntiles == 0) return best;
    const size_t lower = (ntiles + W - 1) / W;
    for (unsigned seed = 0; seed < 64; ++seed) {
        std::mt19937 rng(seed);
        std::vector<Tile> left;
        for (int j = 0; j < nb; ++j)
            for (int k = j + 1; k < nb; ++k) left.push_back({j, k});
        std::shuffle(left.begin(), left.end(), rng);
        std::vector<int> deg(nb, nb - 1);
        std::vector<std::vector<Tile>> rounds;
        while (!left.empty()) {
            std::vector<Tile> rd;
            std::vector<char> used(nb, 0);
            while ((int)rd.size() < W) {
                int pick = -1, score = -1;
                for (size_t i = 0; i < left.size(); ++i) {
                    const Tile &t = left[i];
                    if (used[t.jb] || used[t.kb]) continue;
                    const int s = deg[t.jb] + deg[t.kb];
                    if (s > score) score = s, pick = (int)i;
                }
                if (pick < 0) break;
                const Tile t = left[pick];
                left.erase(left.begin() + pick);
                used[t.jb] = used[t.kb] = 1;
                --deg[t.jb], --deg[t.kb];
                rd.push_back(t);
            }
            rounds.push_back(rd);
        }
        if (best.empty() || rounds.size() < best.size()) best = rounds;
        if (best.size() == lower) break;
    }
    return best;
}

}  // namespace

TransportPlanOffsets build_transport_plan(const crf_tables *t, BlockBuilder &b)
{
    TransportPlanOffsets o;
    const int Ns = t->Ns;
    if (Ns < 17) return o;  // small mechanisms: generic kernel (a register-resident variant is the plan)
    const int nb = (Ns + 7) / 8, NsP = 8 * nb;
    // warps per 32 points: enough warps per SM (>= 12 where the tile count allows), limited by
    // 227 KB of shared memory per SM and by rounds needing W disjoint tiles (2W <= nb)
    const size_t smem32 = sizeof(double) * 2 * (size_t)NsP * 32;
    const int blocks_sm = (int)std::min<size_t>(12, (227 * 1024) / (smem32 + 1024 + 4 * 4 * 32 * 8));
    int W = 1;
    while (W < 4 && blocks_sm * W < 12 && 2 * (2 * W) <= nb) W *= 2;
    o.W = W, o.NsP = NsP, o.nb = nb;

    const int npair = Ns * (Ns + 1) / 2;
    auto pair_index = [&](int j, int k) {
        if (j > k) std::swap(j, k);
        return j * Ns - (j * (j - 1)) / 2 + (k - j);
    };
    auto put_pair = [&](std::vector<double> &dst, int j, int k) {
        for (int c = 0; c < 4; ++c)
            dst.push_back(j < Ns && k < Ns ? -crf::kLog2e * t->D_c[(size_t)c * npair + pair_index(j, k)] : 0.0);
    };
    std::vector<int2> sched;
    std::vector<double> coef;
    auto rounds = schedule_offdiag(nb, W);
    for (auto &rd : rounds)
        for (int w = 0; w < W; ++w) {
            if (w >= (int)rd.size()) {
                sched.push_back(make_int2(0, 0));
                continue;
            }
            const Tile &tl = rd[w];
            sched.push_back(make_int2(1 | tl.jb << 8 | tl.kb << 16, (int)coef.size()));
            for (int a = 0; a < 8; ++a)
                for (int c = 0; c < 8; ++c) put_pair(coef, 8 * tl.jb + a, 8 * tl.kb + c);
        }
    for (int j0 = 0; j0 < nb; j0 += W)
        for (int w = 0; w < W; ++w) {
            const int jb = j0 + w;
            if (jb >= nb) {
                sched.push_back(make_int2(0, 0));
                continue;
            }
            sched.push_back(make_int2(2 | jb << 8 | jb << 16, (int)coef.size()));
            for (int a = 0; a < 8; ++a)
                for (int c = a + 1; c < 8; ++c) put_pair(coef, 8 * jb + a, 8 * jb + c);
        }
    o.n_rounds = (int)(sched.size() / W);

    std::vector<double> cP((size_t)NsP * NsP, 0.0), sp((size_t)NsP * 12, 0.0), dd((size_t)Ns * 4);
    for (int k = 0; k < Ns; ++k) {
        for (int j = 0; j < Ns; ++j) cP[(size_t)k * NsP + j] = 1.0 / std::sqrt(8.0 * (1.0 + t->W[k] / t->W[j]));
        double *s = sp.data() + 12 * (size_t)k;
        for (int c = 0; c < 4; ++c) {
            s[c] = 0.5 * t->mu_c[(size_t)c * Ns + k];
            s[4 + c] = t->lam_c[(size_t)c * Ns + k];
            dd[4 * (size_t)k + c] = t->D_c[(size_t)c * npair + pair_index(k, k)];
        }
        s[8] = 1.0 / std::sqrt(std::sqrt(t->W[k]));
        s[9] = std::sqrt(t->W[k]);
        s[10] = 1.0 / t->W[k];
    }
    o.sched = b.add(sched), o.pair_coef = b.add(coef), o.wilke_cP = b.add(cP), o.sp = b.add(sp), o.Ddiag = b.add(dd);
    return o;
}
