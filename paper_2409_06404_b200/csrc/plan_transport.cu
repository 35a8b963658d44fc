// plan_transport.cu -- host code: the tile schedule and the schedule-ordered tables of
// transport_tiled.cu (see the header comment there and TransportPlan in crf_internal.h).
#include <cmath>
#include <cstdint>

#include "fastmath.cuh"
#include "host_plan.h"

namespace {

struct Tile {
    int kind, jb, kb;  // kind 1: off-diagonal tile (jb < kb), 2: diagonal tile (jb = kb)
};

// Rounds of at most W tiles whose species blocks are pairwise disjoint: the circle method of a round-robin
// tournament over the nb blocks (an odd nb gets a dummy block; meeting the dummy is the block's bye, in
// which it does its own diagonal tile).  nb odd: nb rounds of (nb-1)/2 off-diagonal tiles + 1 diagonal tile
// cover the whole triangle; nb even: nb-1 rounds of nb/2 tiles, then the diagonal tiles.  Rounds with more
// than W tiles are split.
std::vector<std::vector<Tile>> schedule_rounds(int nb, int W)
{
    std::vector<std::vector<Tile>> rounds;
    auto emit = [&](const std::vector<Tile> &tiles) {
        for (size_t i = 0; i < tiles.size(); i += W)
            rounds.emplace_back(tiles.begin() + i, tiles.begin() + std::min(tiles.size(), i + (size_t)W));
    };
    const int ne = nb + (nb & 1), m = ne - 1;  // m rotating blocks, block m is fixed (the dummy when nb is odd)
    for (int r = 0; r < m && nb > 1; ++r) {
        std::vector<Tile> tiles;
        for (int i = 1; i < ne / 2; ++i) {
            const int a = (r + i) % m, c = (r - i + m) % m;
            tiles.push_back({1, std::min(a, c), std::max(a, c)});
        }
        if (nb & 1)
            tiles.push_back({2, r, r});
        else
            tiles.push_back({1, r, m});
        emit(tiles);
    }
    if (!(nb & 1) || nb == 1) {
        std::vector<Tile> tiles;
        for (int j = 0; j < nb; ++j) tiles.push_back({2, j, j});
        emit(tiles);
    }
    return rounds;
}

}  // namespace

TransportPlanOffsets build_transport_plan(const crf_tables *t, const crf_plan_options &opt, BlockBuilder &b)
{
    TransportPlanOffsets o;
    const int Ns = t->Ns;
    const int want = opt.transport_kernel;
    if (want == CRF_TRANSPORT_GENERIC) return o;
    if (Ns < 17) {  // small mechanisms: the register-resident kernel (transport_small.cu), one flat table
        if (Ns < 2 || want == CRF_TRANSPORT_TILED) return o;  // generic kernel (or an unsupported request)
        const int npair = Ns * (Ns + 1) / 2;
        auto pidx = [&](int j, int k) { return j * Ns - (j * (j - 1)) / 2 + (k - j); };  // j <= k
        std::vector<double> tb;
        for (int k = 0; k < Ns; ++k) {
            double s[12] = {0};
            for (int c = 0; c < 4; ++c) {
                s[c] = -0.5 * crf::kLog2e * t->mu_c[(size_t)c * Ns + k];
                s[4 + c] = crf::kLog2e * t->lam_c[(size_t)c * Ns + k];
            }
            s[8] = std::sqrt(std::sqrt(t->W[k])), s[9] = std::sqrt(t->W[k]), s[10] = 1.0 / t->W[k];
            tb.insert(tb.end(), s, s + 12);
        }
        for (int k = 0; k < Ns; ++k)
            for (int c = 0; c < 4; ++c) tb.push_back(t->D_c[(size_t)c * npair + pidx(k, k)]);
        for (int k = 0; k < Ns; ++k)
            for (int j = 0; j < Ns; ++j) tb.push_back(1.0 / std::sqrt(8.0 * (1.0 + t->W[k] / t->W[j])));
        if (tb.size() & 1) tb.push_back(0.0);  // pair fits are read as double2
        for (int j = 0; j < Ns; ++j)
            for (int k = j + 1; k < Ns; ++k)
                for (int c = 0; c < 4; ++c) tb.push_back(-crf::kLog2e * t->D_c[(size_t)c * npair + pidx(j, k)]);
        o.small_n = (int)tb.size();
        o.small = b.add(tb);
        return o;
    }
    if (want == CRF_TRANSPORT_SMALL) return o;  // unsupported request: Ns > 16
    // warps per point group: one per tile of a round-robin round over the nbp pair blocks (nbp odd: (nbp+1)/2, nbp even:
    // nbp/2), at most 8; points per lane: 1 (16 warps per SM at 128 registers) or 2 (8 warps per SM, every coefficient
    // load serves two points).  crf_plan_options.transport_W / transport_PPL override.
    auto warps_for = [&](int nbp) {
        int W = opt.transport_W;
        if (W != 1 && W != 2 && W != 4 && W != 8) {
            const int per_round = std::max(1, (nbp + (nbp & 1)) / 2);
            W = 1;
            while (W < 8 && W < per_round) W *= 2;
            if (nbp <= 3) W = 1;  // a round of nbp = 3 is one full tile and one diagonal tile: two warps would idle 28 %
                                  // (C3: W = 1 3.0 ms, W = 2 4.1 ms); the state is small, so the SM still holds 16 blocks
        }
        return W;
    };
    // Tile edge of the pair phase: 8, or 7 where blocks of 7 species waste fewer padded pairs and idle warps (21 species:
    // three 7-blocks hold exactly the 210 pairs, three 8-blocks evaluate 276; 53 species: eight 7-blocks make full rounds of
    // four tiles, seven 8-blocks leave a warp with the half-size diagonal tile in every round).  The estimate is the
    // warp-time of a point group: W (13 x the largest tile of every round + 3 x the Wilke terms of a warp).
    auto cost_of = [&](int ts) {
        const int nbp = (Ns + ts - 1) / ts, W = warps_for(nbp);
        long pairs = 0;
        for (auto &rd : schedule_rounds(nbp, W)) {
            int worst = 0;
            for (const Tile &tl : rd) worst = std::max(worst, tl.kind == 1 ? ts * ts : ts * (ts - 1) / 2);
            pairs += worst;
        }
        const long wilke = (long)((nbp + W - 1) / W) * ts * ((ts * nbp + 3) / 4 * 4);
        return W * (13 * pairs + 3 * wilke);
    };
    int TS = opt.transport_TS;
    if (TS != 7 && TS != 8) TS = cost_of(7) < cost_of(8) ? 7 : 8;
    // nb blocks of TS species (both phases); the state has NsP rows, all zero past Ns: the Wilke panels read their columns
    // in groups of four and may run up to three rows past the last block
    const int nb = (Ns + TS - 1) / TS, nbp = nb;
    const int W = warps_for(nbp);
    const int PPL = opt.transport_PPL == 2 ? 2 : 1;
    // Wilke panels: up to kPanel column blocks (as many as keep a stage block within 20 KB: fewer, larger stage steps measured
    // faster, C5 panel 3 -> 5 29.2 -> 28.8 ms, C4 15.5 -> 15.0 ms; crf_plan_options.transport_panel overrides)
    const int kPanel = opt.transport_panel > 0 ? std::min(opt.transport_panel, nb) : std::max(1, std::min({nb, 5, 20480 / (W * 512)}));
    int NsP = TS * nb;
    for (int J0 = 0; J0 < nb; J0 += kPanel) NsP = std::max(NsP, TS * J0 + (TS * std::min(kPanel, nb - J0) + 3) / 4 * 4);
    NsP += NsP & 1;
    o.W = W, o.PPL = PPL, o.NsP = NsP, o.nb = nb, o.TS = TS, o.nbp = nbp;

    const int npair = Ns * (Ns + 1) / 2;
    auto pair_index = [&](int j, int k) {
        if (j > k) std::swap(j, k);
        return j * Ns - (j * (j - 1)) / 2 + (k - j);
    };
    auto put_pair = [&](std::vector<double> &dst, int j, int k) {
        for (int c = 0; c < 4; ++c)
            dst.push_back(j < Ns && k < Ns ? -crf::kLog2e * t->D_c[(size_t)c * npair + pair_index(j, k)] : 0.0);
    };
    // Stage blocks (Wilke panels first, then the pair rounds).  Every block starts with a header of
    // hdr = 16 + 8 W (rounded up to 16) bytes: int4 descriptor of the NEXT block {byte offset in pair_coef, bytes,
    // flags, nJ} and, in pair rounds, int2 sched[W] {kind | jb << 8 | kb << 16, byte offset of the tile's
    // coefficients from the block start}: the kernel's loops read no descriptor from global memory.
    const size_t hdr_d = (16 + 8 * (size_t)W + 15) / 16 * 2;  // header size in doubles
    std::vector<int4> rdesc;
    std::vector<double> coef;
    size_t stage_bytes = 16;
    auto put_i = [&](size_t byte_off, int v) { std::memcpy(reinterpret_cast<unsigned char *>(coef.data()) + byte_off, &v, 4); };
    auto close_block = [&](size_t start, int flags, int nJ) {
        if (coef.size() & 1) coef.push_back(0.0);
        rdesc.push_back(make_int4((int)(8 * start), (int)(8 * (coef.size() - start)), flags, nJ));
        stage_bytes = std::max(stage_bytes, 8 * (coef.size() - start));
    };
    // Wilke stage blocks: pass p covers the row blocks p W .. p W + W - 1 (one per warp), a panel covers up to kPanel column
    // blocks; payload [W][TS rows][ld columns] of c_kj (0 in padded rows/columns), ld = TS nJ rounded up to a multiple of 4;
    // descriptor w = nJ
    const int npass = (nb + W - 1) / W;
    for (int ps = 0; ps < npass; ++ps)
        for (int J0 = 0; J0 < nb; J0 += kPanel) {
            const int nJ = std::min(kPanel, nb - J0);
            const size_t start = coef.size();
            coef.resize(start + hdr_d, 0.0);
            const int ld = (TS * nJ + 3) / 4 * 4;
            for (int w = 0; w < W; ++w)
                for (int a = 0; a < TS; ++a)
                    for (int c = 0; c < ld; ++c) {
                        const int k = TS * (ps * W + w) + a, j = TS * J0 + c;
                        coef.push_back(c < TS * nJ && k < Ns && j < Ns ? 1.0 / std::sqrt(8.0 * (1.0 + t->W[k] / t->W[j])) : 0.0);
                    }
            close_block(start, J0 | ps << 8 | (J0 == 0) << 16 | (J0 + nJ == nb) << 17, nJ);
        }
    o.n_wilke = (int)rdesc.size();
    for (auto &rd : schedule_rounds(nbp, W)) {
        const size_t start = coef.size();
        coef.resize(start + hdr_d, 0.0);
        for (int w = 0; w < (int)rd.size(); ++w) {
            const Tile &tl = rd[w];
            put_i(8 * start + 16 + 8 * (size_t)w, tl.kind | tl.jb << 8 | tl.kb << 16);
            put_i(8 * start + 16 + 8 * (size_t)w + 4, (int)(8 * (coef.size() - start)));
            for (int a = 0; a < TS; ++a)
                for (int c = tl.kind == 1 ? 0 : a + 1; c < TS; ++c) put_pair(coef, TS * tl.jb + a, TS * tl.kb + c);
        }
        close_block(start, 0, 0);
    }
    o.n_rounds = (int)rdesc.size() - o.n_wilke;
    o.stage_bytes = (int)stage_bytes;
    for (size_t i = 0; i + 1 < rdesc.size(); ++i) {
        const int4 nx = rdesc[i + 1];
        put_i((size_t)rdesc[i].x + 0, nx.x), put_i((size_t)rdesc[i].x + 4, nx.y);
        put_i((size_t)rdesc[i].x + 8, nx.z), put_i((size_t)rdesc[i].x + 12, nx.w);
    }

    std::vector<double> cP((size_t)NsP * NsP, 0.0), sp((size_t)NsP * 12, 0.0), dd((size_t)Ns * 4);
    for (int k = 0; k < Ns; ++k) {
        for (int j = 0; j < Ns; ++j) cP[(size_t)k * NsP + j] = 1.0 / std::sqrt(8.0 * (1.0 + t->W[k] / t->W[j]));
        double *s = sp.data() + 12 * (size_t)k;
        for (int c = 0; c < 4; ++c) {
            s[c] = -0.5 * crf::kLog2e * t->mu_c[(size_t)c * Ns + k];
            s[4 + c] = crf::kLog2e * t->lam_c[(size_t)c * Ns + k];
            dd[4 * (size_t)k + c] = t->D_c[(size_t)c * npair + pair_index(k, k)];
        }
        s[8] = std::sqrt(std::sqrt(t->W[k]));
        s[9] = std::sqrt(t->W[k]);
        s[10] = 1.0 / t->W[k];
    }
    o.rounds = b.add(rdesc), o.pair_coef = b.add(coef), o.wilke_cP = b.add(cP), o.sp = b.add(sp), o.Ddiag = b.add(dd);
    return o;
}

extern "C" int crf_transport_schedule(int nb, int W, int32_t *out, int cap)
{
    if (nb < 1 || nb > 255 || W < 1 || W > 8 || (cap > 0 && !out)) return CRF_EINVAL;
    int count = 0, rd = 0;
    for (auto &round : schedule_rounds(nb, W)) {
        for (const Tile &tl : round) {
            if (count < cap) {
                int32_t *o = out + 4 * (size_t)count;
                o[0] = rd, o[1] = tl.kind, o[2] = tl.jb, o[3] = tl.kb;
            }
            ++count;
        }
        ++rd;
    }
    return count;
}
