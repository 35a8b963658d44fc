// plan_rates_smem.cu -- host code: chunk blocks of rates_smem.cu (layout in RatesSmemPlan, crf_internal.h),
// the choice of warps per point group / points per lane / chunk size from the shared-memory budget, and
// the range check that admits the product form of the equilibrium constant.
#include <cmath>
#include <cstdint>

#include "fastmath.cuh"
#include "host_plan.h"

namespace {

struct Builder {
    const crf_tables *t;
    int Ns, Nr, N3, Nt, Ne;
    int slot(const int16_t *tab, int s, int r) const { return (int)tab[(size_t)s * Nr + r]; }
    bool generic(int r) const { return slot(t->reac, 2, r) >= 0 || slot(t->prod, 2, r) >= 0; }
    int kind(int r) const { return r < Ne ? 0 : (r < Ne + N3 ? 1 : 2); }
};

template <class T>
void put(std::vector<unsigned char> &v, size_t off, const T &x)
{
    std::memcpy(v.data() + off, &x, sizeof(T));
}

// log2(e) g_k/(RT) of species k at temperature T (the value the kernel's state is built from)
double gamma2(const crf_tables *t, int k, double T)
{
    const int Ns = t->Ns;
    const double *a = T <= t->Tmid[k] ? t->nasa_lo : t->nasa_hi;
    auto A = [&](int c) { return a[(size_t)c * Ns + k]; };
    const double h = A(0) + T * (A(1) / 2 + T * (A(2) / 3 + T * (A(3) / 4 + T * A(4) / 5))) + A(5) / T;
    const double s = A(0) * std::log(T) + T * (A(1) + T * (A(2) / 2 + T * (A(3) / 3 + T * A(4) / 4))) + A(6);
    return crf::kLog2e * (h - s);
}

// The kernel forms 1/K_c = (d_a0 d_a1 [d_a2]) / (d_b0 d_b1 [d_b2]) with d_k = (p_ref/RT) 2^(-gamma_k): numerator,
// denominator and quotient must stay far inside the double range for every T the path is specified for.
bool product_form_in_range(const Builder &B)
{
    const crf_tables *t = B.t;
    const int NT = 96;
    const double Tlo = 250.0, Thi = 5000.0, limit = 960.0;
    std::vector<double> l2d((size_t)B.Ns);
    for (int it = 0; it < NT; ++it) {
        const double T = Tlo * std::pow(Thi / Tlo, it / double(NT - 1));
        const double l2c0 = std::log2(t->p_ref / (CRF_R_GAS * T));
        for (int k = 0; k < B.Ns; ++k) l2d[k] = l2c0 - gamma2(t, k, T);
        for (int r = 0; r < B.Nr; ++r) {
            double num = 0.0, den = 0.0;
            for (int s = 0; s < 3; ++s) {
                const int a = B.slot(t->reac, s, r), b = B.slot(t->prod, s, r);
                if (a >= 0) num += l2d[a];
                if (b >= 0) den += l2d[b];
            }
            if (!(std::fabs(num) < limit && std::fabs(den) < limit && std::fabs(num - den) < limit)) return false;
        }
    }
    return true;
}

struct Chunk {
    int kind, generic;
    std::vector<int> reactions;
};

std::vector<Chunk> make_chunks(const Builder &B, int Rc)
{
    std::vector<Chunk> out;
    for (int kind = 0; kind < 3; ++kind)
        for (int g = 0; g < 2; ++g) {
            std::vector<int> grp;
            for (int r = 0; r < B.Nr; ++r)
                if (B.kind(r) == kind && (int)B.generic(r) == g) grp.push_back(r);
            if (grp.empty()) continue;
            const int nch = ((int)grp.size() + Rc - 1) / Rc;
            for (int c = 0; c < nch; ++c) {  // equal shares
                const size_t lo = grp.size() * c / nch, hi = grp.size() * (c + 1) / nch;
                Chunk ch{kind, g, std::vector<int>(grp.begin() + lo, grp.begin() + hi)};
                out.push_back(ch);
            }
        }
    return out;
}

std::vector<unsigned char> chunk_block(const Builder &B, const Chunk &ch, int PPL, int W, int maxown)
{
    const crf_tables *t = B.t;
    const int Ns = B.Ns, cnt = (int)ch.reactions.size();
    const unsigned row = 512u * PPL;   // bytes per species row of the (C, d) state
    const unsigned qrow = 256u * PPL;  // bytes per reaction row of the q buffer
    const size_t o_slot = 48 * (size_t)cnt;
    const size_t slot_row = 16 + 4 * (size_t)maxown;  // per warp: start, 3 pad words, end of each owned slot
    const size_t o_troe = o_slot + slot_row * W;
    size_t o_list = o_troe + (ch.kind == 2 ? 64 * (size_t)cnt : 0);
    std::vector<unsigned char> v(o_list, 0);
    auto row_of = [&](int k) { return (unsigned)(k >= 0 ? k : Ns) * row; };  // row Ns: the dummy species (1, 1)
    auto append16 = [&](double x, unsigned y) {
        const size_t o = v.size();
        v.resize(o + 16, 0);
        put(v, o, x);
        put(v, o + 8, y);
        return o;
    };
    // incidence entries: warp-major, then the warp's owned species k = w + W s in slot order
    for (int w = 0; w < W; ++w) {
        put(v, o_slot + slot_row * w, (unsigned)v.size());
        for (int sl = 0; sl < maxown; ++sl) {
            const int k = w + W * sl;
            int cnt_slot = 0;
            for (int rl = 0; rl < cnt && k < Ns; ++rl) {
                const int r = ch.reactions[rl];
                int nu = 0;
                for (int s = 0; s < 3; ++s) nu += (B.slot(t->prod, s, r) == k) - (B.slot(t->reac, s, r) == k);
                if (nu != 0) append16((double)nu, (unsigned)rl * qrow), ++cnt_slot;
            }
            if (cnt_slot & 1) append16(0.0, 0u);  // the entry loop takes two entries per trip
            put(v, o_slot + slot_row * w + 16 + 4 * (size_t)sl, (unsigned)v.size());
        }
    }
    append16(0.0, 0u), append16(0.0, 0u);  // the entry loop reads two entries ahead
    for (int rl = 0; rl < cnt; ++rl) {
        const int r = ch.reactions[rl];
        const size_t o = 48 * (size_t)rl;
        put(v, o + 0, crf::kLog2e * t->lnA[r]);
        put(v, o + 8, crf::kLog2e * t->beta[r]);
        put(v, o + 16, -crf::kLog2e * t->Ea_R[r]);
        unsigned x0 = row_of(B.slot(t->reac, 2, r)), x1 = row_of(B.slot(t->prod, 2, r));
        if (ch.kind != 0) {
            const int mrow = r - B.Ne;
            x0 = (unsigned)v.size();
            x1 = (unsigned)(t->eff_ptr[mrow + 1] - t->eff_ptr[mrow]);
            for (int e = t->eff_ptr[mrow]; e < t->eff_ptr[mrow + 1]; ++e) append16(t->eff_val[e], row_of(t->eff_idx[e]));
        }
        put(v, o + 24, x0);
        put(v, o + 28, x1);
        put(v, o + 32, row_of(B.slot(t->reac, 0, r)));
        put(v, o + 36, row_of(B.slot(t->reac, 1, r)));
        put(v, o + 40, row_of(B.slot(t->prod, 0, r)));
        put(v, o + 44, row_of(B.slot(t->prod, 1, r)));
        if (ch.kind == 2) {
            const int i = r - B.Ne - B.N3;
            const double q[8] = {crf::kLog2e * t->lnA0[i], crf::kLog2e * t->beta0[i], -crf::kLog2e * t->Ea0_R[i],
                                 t->alpha[i],              -crf::kLog2e / t->T3[i], -crf::kLog2e / t->T1[i],
                                 -crf::kLog2e * t->T2[i],  0.0};
            std::memcpy(v.data() + o_troe + 64 * (size_t)rl, q, sizeof(q));
        }
    }
    return v;
}

}  // namespace

RatesSmemPlanOffsets build_rates_smem_plan(const crf_tables *t, const crf_plan_options &opt, BlockBuilder &b)
{
    RatesSmemPlanOffsets o;
    Builder B{t, t->Ns, t->Nr, t->N3, t->Nt, t->Nr - t->N3 - t->Nt};
    const int Ns = B.Ns, Nr = B.Nr;
    const int want = opt.rates_kernel;
    if (Nr == 0 || Ns > 256 || want == CRF_RATES_STAGED || want == CRF_RATES_GENERIC || want == CRF_RATES_GROUP) return o;
    for (int r = B.Ne; r < Nr; ++r)
        if (B.generic(r)) return o;  // a third body next to three explicit reactants: staged kernel
    if (!product_form_in_range(B)) return o;

    std::vector<Chunk> chunks;
    std::vector<std::vector<unsigned char>> blocks;
    size_t stage_bytes = 0;
    // Small mechanisms: one THREAD per point (rates_thread_kernel in rates_smem.cu), 128 points per block, the (C, d)
    // state and omega as per-thread columns in shared memory (row stride 128 x 16 bytes = the layout of "4 points
    // per lane"), all chunk blocks resident at once.  Marked W = 1, PPL = 4; stage_bytes = all blocks.
    // Default for Ns <= 12 (C2: 2.96 ms against 3.40 ms for the warp-group kernel); on request (CRF_RATES_THREAD) up to
    // Ns = 24 (C3: 3.9 against 2.4 ms: the per-thread shared-memory chains are not hidden at 12 warps per SM).
    if (Ns <= 24 && (want == CRF_RATES_THREAD || (want == CRF_RATES_AUTO && Ns <= 12 && opt.rates_W == 0))) {
        chunks = make_chunks(B, Nr);
        for (const Chunk &ch : chunks) {
            blocks.push_back(chunk_block(B, ch, 4, 1, 4));
            stage_bytes += (blocks.back().size() + 15) & ~size_t(15);
        }
        if (stage_bytes <= 24 * 1024) o.W = 1, o.PPL = 4, o.maxown = 4, o.Rc = 0;
    }
    if (o.W == 0) return o;  // (larger mechanisms: rates_group.cu)
    if (chunks.size() > 64) return RatesSmemPlanOffsets();  // the kernel keeps at most 64 chunk descriptors
    o.n_chunks = (int)chunks.size(), o.stage_bytes = (int)stage_bytes;

    std::vector<int4> cdesc;
    std::vector<unsigned char> stage;
    for (size_t c = 0; c < chunks.size(); ++c) {
        const size_t off = stage.size();
        stage.insert(stage.end(), blocks[c].begin(), blocks[c].end());
        stage.resize((stage.size() + 15) & ~size_t(15), 0);
        cdesc.push_back(make_int4(chunks[c].kind | chunks[c].generic << 2, (int)chunks[c].reactions.size(), (int)off,
                                  (int)(stage.size() - off)));
    }
    stage.resize(stage.size() + stage_bytes, 0);  // the copy of a block may run to stage_bytes: keep it in bounds

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
    o.chunk = b.add(cdesc), o.stage = b.add(stage), o.gco = b.add(gco), o.hco = b.add(hco);
    return o;
}
