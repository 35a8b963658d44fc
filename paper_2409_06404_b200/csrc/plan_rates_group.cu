// plan_rates_group.cu -- host code: the chunk blocks of rates_group.cu (layout in RatesGroupPlan, crf_internal.h),
// the choice of warps per point group / points per lane / chunk size from the shared-memory budget, the
// balanced deal of reactions to warps and of species to owners, and the range check that admits the
// activity form of the rate of progress.
#include <cmath>
#include <cstdint>
#include <numeric>

#include "fastmath.cuh"
#include "host_plan.h"

namespace {

struct Mech {
    const crf_tables *t;
    int Ns, Nr, N3, Nt, Ne;
    int slot(const int16_t *tab, int s, int r) const { return (int)tab[(size_t)s * Nr + r]; }
    bool generic(int r) const { return slot(t->reac, 2, r) >= 0 || slot(t->prod, 2, r) >= 0; }
    int kind(int r) const { return r < Ne ? 0 : (r < Ne + N3 ? 1 : 2); }
    int n_eff(int r) const { return r < Ne ? 0 : t->eff_ptr[r - Ne + 1] - t->eff_ptr[r - Ne]; }
    // net stoichiometric coefficient of species k in reaction r
    int nu(int r, int k) const
    {
        int v = 0;
        for (int s = 0; s < 3; ++s) v += (slot(t->prod, s, r) == k) - (slot(t->reac, s, r) == k);
        return v;
    }
    // relative cost of one reaction in the reaction stage (FP64 + shared-memory work; an elementary reaction = 1)
    double cost(int r) const
    {
        const double base = kind(r) == 2 ? 7.0 : (kind(r) == 1 ? 1.15 : 1.0);
        return base + (generic(r) ? 0.25 : 0.0) + 0.22 * n_eff(r);
    }
};

template <class T>
void put(std::vector<unsigned char> &v, size_t off, const T &x)
{
    std::memcpy(v.data() + off, &x, sizeof(T));
}

// log2 d_k(T), d_k = (p_ref/RT) exp(-g_k/RT): the per-species factor the kernel's state is built from
double log2_d(const crf_tables *t, int k, double T)
{
    const int Ns = t->Ns;
    const double *a = T <= t->Tmid[k] ? t->nasa_lo : t->nasa_hi;
    auto A = [&](int c) { return a[(size_t)c * Ns + k]; };
    const double h = A(0) + T * (A(1) / 2 + T * (A(2) / 3 + T * (A(3) / 4 + T * A(4) / 5))) + A(5) / T;
    const double s = A(0) * std::log(T) + T * (A(1) + T * (A(2) / 2 + T * (A(3) / 3 + T * A(4) / 4))) + A(6);
    return std::log2(t->p_ref / (CRF_R_GAS * T)) - crf::kLog2e * (h - s);
}

// The kernel evaluates q = k_f prod_reactants d_a (prod_reactants u_a - prod_products u_b), u_k = C_k / d_k
// (rates_group.cu).  Every factor must stay a normal double for every T in [250, 5000] K and every concentration
// between kCmin and kCmax kmol/m^3 (an exact zero is fine); otherwise the log-space kernel runs.
bool activity_form_in_range(const Mech &B)
{
    const crf_tables *t = B.t;
    const int NT = 96;
    const double Tlo = 250.0, Thi = 5000.0, limit = 1000.0;
    const double l2Cmin = std::log2(1.0e-36), l2Cmax = std::log2(1.0e4);
    std::vector<double> l2d((size_t)B.Ns);
    for (int it = 0; it < NT; ++it) {
        const double T = Tlo * std::pow(Thi / Tlo, it / double(NT - 1)), L = std::log(T);
        for (int k = 0; k < B.Ns; ++k) {
            l2d[k] = log2_d(t, k, T);
            if (!(std::fabs(l2d[k]) < limit)) return false;
        }
        for (int r = 0; r < B.Nr; ++r) {
            double sa = 0.0, sb = 0.0;
            int na = 0, nb = 0;
            for (int s = 0; s < 3; ++s) {
                const int a = B.slot(t->reac, s, r), b = B.slot(t->prod, s, r);
                if (a >= 0) sa += l2d[a], ++na;
                if (b >= 0) sb += l2d[b], ++nb;
            }
            const double y = crf::kLog2e * (t->lnA[r] + t->beta[r] * L - t->Ea_R[r] / T);  // log2 k_f
            // prod d_a, k_f prod d_a, prod u_a, prod u_b (largest and smallest magnitude each can take)
            if (!(std::fabs(sa) < limit && std::fabs(y) < limit && std::fabs(y + sa) < limit)) return false;
            if (!(-sa + na * l2Cmin > -limit && -sa + na * l2Cmax < limit)) return false;
            if (!(-sb + nb * l2Cmin > -limit && -sb + nb * l2Cmax < limit)) return false;
        }
    }
    return true;
}

struct WarpList {
    std::vector<int> rx;  // reactions in processing order: elementary, elementary with three slots, third body, falloff
    double load = 0.0;
};

struct Chunk {
    std::vector<int> rx;          // all reactions of the chunk
    std::vector<WarpList> warps;  // dealt to the W warps
};

int order_key(const Mech &B, int r) { return B.kind(r) * 2 + (B.kind(r) == 0 && B.generic(r) ? 1 : 0); }

// Reactions -> chunks -> warps.  Chunks get equal counts and, as far as the counts allow, equal cost (the expensive
// kinds are dealt round-robin); inside a chunk the reactions go, most expensive first, to the least loaded warp.
std::vector<Chunk> make_chunks(const Mech &B, int n_chunks, int W)
{
    std::vector<int> order(B.Nr);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return B.cost(a) > B.cost(b); });
    std::vector<Chunk> ch((size_t)n_chunks);
    for (int i = 0; i < B.Nr; ++i) ch[(size_t)(i % n_chunks)].rx.push_back(order[i]);
    for (Chunk &c : ch) {
        c.warps.assign((size_t)W, WarpList());
        for (int r : c.rx) {  // (already sorted by decreasing cost)
            size_t best = 0;
            for (size_t w = 1; w < c.warps.size(); ++w)
                if (c.warps[w].load < c.warps[best].load) best = w;
            c.warps[best].rx.push_back(r);
            c.warps[best].load += B.cost(r);
        }
        for (WarpList &wl : c.warps)
            std::stable_sort(wl.rx.begin(), wl.rx.end(), [&](int a, int b) { return order_key(B, a) < order_key(B, b); });
    }
    return ch;
}

// Species -> (warp, slot), balanced by the number of incidence entries (species with the most reactions first, each
// to the least loaded warp that still has a free slot).
std::vector<int> deal_species(const Mech &B, int W, int maxown)
{
    std::vector<int> deg((size_t)B.Ns, 0), order((size_t)B.Ns);
    for (int r = 0; r < B.Nr; ++r)
        for (int k = 0; k < B.Ns; ++k) deg[k] += std::abs(B.nu(r, k));
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return deg[a] > deg[b]; });
    std::vector<int> own((size_t)W * maxown, -1), used((size_t)W, 0), load((size_t)W, 0);
    for (int k : order) {
        int best = -1;
        for (int w = 0; w < W; ++w)
            if (used[w] < maxown && (best < 0 || load[w] < load[best] || (load[w] == load[best] && used[w] < used[best])))
                best = w;
        own[(size_t)best * maxown + used[best]++] = k;
        load[best] += deg[k] + 2;  // (+2: the prologue / epilogue work every owned species costs)
    }
    return own;
}

// One chunk block (layout: RatesGroupPlan in crf_internal.h)
std::vector<unsigned char> chunk_block(const Mech &B, const Chunk &ch, const std::vector<int> &own, int PPL, int W,
                                       int maxown, int Rc, bool tm)
{
    const crf_tables *t = B.t;
    const int Ns = B.Ns;
    const unsigned rowb = 256u * PPL;  // bytes of one row (32 lanes x PPL doubles)
    // d row k: byte offset k rowb in the shared-memory state; u row k: tensor-memory column 2 PPL k, or the shared-memory
    // row Ns + 1 + k; empty slots point at the dummy species, row Ns (u = d = 1)
    auto d_of = [&](int k) { return (unsigned)(k >= 0 ? k : Ns) * rowb; };
    auto u_of = [&](int k) {
        const unsigned kk = (unsigned)(k >= 0 ? k : Ns);
        return tm ? 2u * PPL * kk : (unsigned)(Ns + 1 + kk) * rowb;
    };
    const size_t hdr = 32 * (size_t)W;
    std::vector<unsigned char> v(hdr, 0);
    auto align16 = [&]() { v.resize((v.size() + 15) & ~size_t(15), 0); };
    // q row of every reaction of the chunk: warp-major processing order
    std::vector<int> qrow((size_t)B.Nr, -1);
    int next_row = 0;
    for (int w = 0; w < W; ++w)
        for (int r : ch.warps[w].rx) qrow[r] = next_row++;
    // records (+ Troe sets and third-body lists) per warp
    for (int w = 0; w < W; ++w) {
        const WarpList &wl = ch.warps[w];
        align16();
        const size_t rec0 = v.size();
        v.resize(rec0 + 64 * wl.rx.size(), 0);
        uint16_t cnt[4] = {0, 0, 0, 0};
        size_t troe0 = 0;
        int n_troe = 0;
        for (int r : wl.rx) n_troe += B.kind(r) == 2;
        if (n_troe) {
            troe0 = v.size();
            v.resize(troe0 + 64 * (size_t)n_troe, 0);
        }
        int it = 0;
        for (size_t i = 0; i < wl.rx.size(); ++i) {
            const int r = wl.rx[i];
            ++cnt[B.kind(r) == 0 ? (B.generic(r) ? 1 : 0) : B.kind(r) + 1];
            const size_t o = rec0 + 64 * i;
            put(v, o + 0, crf::kLog2e * t->lnA[r]);
            put(v, o + 8, crf::kLog2e * t->beta[r]);
            put(v, o + 16, -crf::kLog2e * t->Ea_R[r]);
            put(v, o + 24, u_of(B.slot(t->prod, 0, r)));
            put(v, o + 28, u_of(B.slot(t->prod, 1, r)));
            put(v, o + 32, d_of(B.slot(t->reac, 0, r)));
            put(v, o + 36, d_of(B.slot(t->reac, 1, r)));
            put(v, o + 40, u_of(B.slot(t->reac, 0, r)));
            put(v, o + 44, u_of(B.slot(t->reac, 1, r)));
            unsigned x0 = d_of(B.slot(t->reac, 2, r)), x1 = 0;
            if (B.kind(r) != 0) {
                const int mrow = r - B.Ne;
                align16();
                x0 = (unsigned)v.size();
                x1 = (unsigned)(t->eff_ptr[mrow + 1] - t->eff_ptr[mrow]);
                for (int e = t->eff_ptr[mrow]; e < t->eff_ptr[mrow + 1]; ++e) {
                    const size_t eo = v.size();
                    v.resize(eo + 16, 0);
                    put(v, eo, t->eff_val[e]);
                    put(v, eo + 8, d_of(t->eff_idx[e]));
                    put(v, eo + 12, u_of(t->eff_idx[e]));
                }
            }
            put(v, o + 48, x0);
            put(v, o + 52, x1);
            put(v, o + 56, u_of(B.slot(t->reac, 2, r)));
            put(v, o + 60, u_of(B.slot(t->prod, 2, r)));
            if (B.kind(r) == 2) {
                const int i2 = r - B.Ne - B.N3;
                const double q[8] = {crf::kLog2e * t->lnA0[i2], crf::kLog2e * t->beta0[i2], -crf::kLog2e * t->Ea0_R[i2],
                                     t->alpha[i2],              -crf::kLog2e / t->T3[i2], -crf::kLog2e / t->T1[i2],
                                     -crf::kLog2e * t->T2[i2],  0.0};
                std::memcpy(v.data() + troe0 + 64 * (size_t)it++, q, sizeof(q));
            }
        }
        const unsigned q0 = wl.rx.empty() ? 0u : (unsigned)qrow[wl.rx[0]] * rowb;
        put(v, 32 * (size_t)w + 0, (unsigned)rec0);
        put(v, 32 * (size_t)w + 4, q0);
        put(v, 32 * (size_t)w + 12, (unsigned)troe0);
        for (int c = 0; c < 4; ++c) put(v, 32 * (size_t)w + 16 + 2 * (size_t)c, cnt[c]);
    }
    // incidence lists per warp, slot-major: plus list then minus list of each owned species, u32 = byte offset of the q
    // row (|nu| = 2 -> two entries), each list padded to even length with the zero row (row Rc)
    for (int w = 0; w < W; ++w) {
        align16();
        const size_t tab = v.size();
        v.resize(tab + 8 * (size_t)maxown + 16, 0);  // {endP, endM}[maxown], start, pad
        put(v, 32 * (size_t)w + 8, (unsigned)tab);
        put(v, tab + 8 * (size_t)maxown, (unsigned)v.size());
        for (int sl = 0; sl < maxown; ++sl) {
            const int k = own[(size_t)w * maxown + sl];
            for (int sign = +1; sign >= -1; sign -= 2) {
                int cnt = 0;
                if (k >= 0)
                    for (int r : ch.rx) {
                        const int nu = B.nu(r, k);
                        for (int c = 0; c < std::abs(nu) && nu * sign > 0; ++c, ++cnt) {
                            const size_t eo = v.size();
                            v.resize(eo + 4, 0);
                            put(v, eo, (unsigned)qrow[r] * rowb);
                        }
                    }
                if (cnt & 1) {
                    const size_t eo = v.size();
                    v.resize(eo + 4, 0);
                    put(v, eo, (unsigned)Rc * rowb);
                }
                put(v, tab + 8 * (size_t)sl + (sign > 0 ? 0 : 4), (unsigned)v.size());
            }
        }
    }
    align16();
    return v;
}

}  // namespace

RatesGroupPlanOffsets build_rates_group_plan(const crf_tables *t, const crf_plan_options &opt, BlockBuilder &b)
{
    RatesGroupPlanOffsets o;
    Mech B{t, t->Ns, t->Nr, t->N3, t->Nt, t->Nr - t->N3 - t->Nt};
    const int Ns = B.Ns, Nr = B.Nr;
    const int want = opt.rates_kernel;
    if (Nr == 0 || (want != CRF_RATES_AUTO && want != CRF_RATES_GROUP)) return o;
    for (int r = B.Ne; r < Nr; ++r)
        if (B.generic(r)) return o;  // a third body next to three explicit reactants: staged kernel
    if (!activity_form_in_range(B)) return o;

    // Warps per point group W and points per lane PPL.  The register file holds 16 warps of 128 registers per SM, so a
    // block of W warps may use 1/(16/W) of the SM's shared memory.  Two points per lane whenever the state of 64
    // points (2 rows of 512 bytes per species) leaves at least 40 % of that for the q buffer and the chunk tables,
    // and the fewest warps for which that holds (more blocks per SM: their phases interleave).
    auto budget = [](int W) { return (size_t)233472 / (16 / W) - 1024; };
    auto state = [&](int PPL) { return (size_t)(Ns + 1) * 512 * PPL; };
    auto pick_w = [&](int ppl) {
        for (int w = 4; w <= 16; w *= 2)
            if (state(ppl) <= budget(w) * 6 / 10 && (Ns + w - 1) / w <= 16) return w;
        return 0;
    };
    int PPL = opt.rates_PPL ? opt.rates_PPL : (pick_w(2) ? 2 : 1);
    if (PPL != 1 && PPL != 2) return o;
    int W = opt.rates_W;
    if (W != 0 && W != 4 && W != 8 && W != 16) return o;
    if (W == 0) W = pick_w(PPL) ? pick_w(PPL) : 16;
    if ((Ns + W - 1) / W > 16) return o;
    const int own_n = (Ns + W - 1) / W, maxown = own_n <= 4 ? 4 : (own_n <= 8 ? 8 : 16);
    const std::vector<int> own = deal_species(B, W, maxown);

    // U in tensor memory (rates_group.cu): 2 PPL columns per species (+ the dummy species), a power of two >= 32 per
    // block, and the 16/W blocks an SM holds must fit the 512 columns together
    int tm_cols = 32;
    while (tm_cols < 2 * PPL * (Ns + 1)) tm_cols *= 2;
    const bool tm_fits = tm_cols <= 512 && (16 / W) * tm_cols <= 512;
    if (opt.rates_tmem == 2 && !tm_fits) return o;
    const bool tm = opt.rates_tmem == 1 ? false : tm_fits;
    if (!tm) tm_cols = 0;

    // Chunks: as few as the q buffer allows (Rc + 1 rows of 256 PPL bytes next to the state and two stage buffers; with
    // U in tensor memory the prologue also passes the u rows through the q buffer: W + Ns + 1 rows)
    const size_t fixed = (tm ? state(PPL) / 2 : state(PPL)) + 1536;  // + mbarriers, chunk descriptors
    std::vector<Chunk> chunks;
    std::vector<std::vector<unsigned char>> blocks;
    size_t stage_bytes = 0;
    int Rc = 0, q_rows = 0;
    const int first = opt.rates_Rc > 0 ? std::max(1, (Nr + opt.rates_Rc - 1) / opt.rates_Rc) : 1;
    for (int n_chunks = first;; ++n_chunks) {
        if (n_chunks > 64 || n_chunks > Nr) return o;  // does not fit at all
        chunks = make_chunks(B, n_chunks, W);
        Rc = 0;
        for (const Chunk &c : chunks) Rc = std::max(Rc, (int)c.rx.size());
        q_rows = std::max(Rc + 1, tm ? W + Ns + 1 : 3 * W);  // (the epilogue reduces three block-wide sums: 3 W rows)
        q_rows = std::max(q_rows, 3 * W);
        blocks.clear();
        stage_bytes = 0;
        for (const Chunk &c : chunks) {
            blocks.push_back(chunk_block(B, c, own, PPL, W, maxown, Rc, tm));
            stage_bytes = std::max(stage_bytes, blocks.back().size());
        }
        stage_bytes = std::max(stage_bytes, (size_t)128 * Ns);  // the buffers also carry the NASA sets (prologue, epilogue)
        if (fixed + (size_t)q_rows * 256 * PPL + 2 * stage_bytes <= budget(W)) break;
    }
    o.q_rows = q_rows, o.tm_cols = tm_cols;
    o.log2_c0 = std::log2(t->p_ref / CRF_R_GAS);
    o.W = W, o.PPL = PPL, o.maxown = maxown, o.Rc = Rc;
    o.n_chunks = (int)chunks.size(), o.stage_bytes = (int)stage_bytes;

    std::vector<int4> cdesc;
    std::vector<unsigned char> stage;
    for (size_t c = 0; c < chunks.size(); ++c) {
        const size_t off = stage.size();
        stage.insert(stage.end(), blocks[c].begin(), blocks[c].end());
        cdesc.push_back(make_int4((int)off, (int)blocks[c].size(), (int)chunks[c].rx.size(), 0));
    }
    // NASA sets: log2(e) g/(RT) = c0 (1 - ln T) + T (c1 + T (c2 + T (c3 + T c4))) + c5/T + c6 ; h/(RT) plain
    std::vector<double> gco((size_t)Ns * 16, 0.0), hco((size_t)Ns * 16, 0.0);
    for (int k = 0; k < Ns; ++k)
        for (int rg = 0; rg < 2; ++rg) {
            const double *a = rg == 0 ? t->nasa_lo : t->nasa_hi;
            auto A = [&](int c) { return a[(size_t)c * Ns + k]; };
            double *g = gco.data() + 16 * (size_t)k + 8 * rg, *h = hco.data() + 16 * (size_t)k + 8 * rg;
            const double s = crf::kLog2e;
            g[0] = s * A(0), g[1] = -s * A(1) / 2.0, g[2] = -s * A(2) / 6.0, g[3] = -s * A(3) / 12.0,
            g[4] = -s * A(4) / 20.0, g[5] = s * A(5), g[6] = -s * A(6);
            h[0] = A(0), h[1] = A(1) / 2.0, h[2] = A(2) / 3.0, h[3] = A(3) / 4.0, h[4] = A(4) / 5.0, h[5] = A(5);
            if (rg == 0) g[7] = t->Tmid[k], h[7] = t->Tmid[k];
            if (rg == 1) g[7] = 1.0 / t->W[k], h[7] = 1.0 / t->W[k];
        }
    o.chunk = b.add(cdesc), o.stage = b.add(stage), o.gco = b.add(gco), o.hco = b.add(hco), o.own = b.add(own);
    return o;
}
