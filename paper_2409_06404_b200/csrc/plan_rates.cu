// plan_rates.cu -- host code: reaction chunks, per-chunk incidence lists and re-laid-out coefficient
// tables of rates_staged.cu (see the header comment there and RatesPlan in crf_internal.h).
#include <cmath>
#include <cstdint>

#include "fastmath.cuh"
#include "host_plan.h"

RatesPlanOffsets build_rates_plan(const crf_tables *t, const crf_plan_options &opt, BlockBuilder &b)
{
    RatesPlanOffsets o;
    const int Ns = t->Ns, Nr = t->Nr, N3 = t->N3, Nt = t->Nt, Ne = Nr - N3 - Nt;
    if (Ns > 128 || Nr == 0) return o;  // owned-species accumulators are registers: at most 32 per warp
    if (opt.rates_kernel != CRF_RATES_AUTO && opt.rates_kernel != CRF_RATES_STAGED) return o;
    int W = Ns >= 32 ? 4 : (Ns >= 12 ? 2 : 1);
    if (opt.rates_kernel == CRF_RATES_STAGED && (opt.rates_W == 1 || opt.rates_W == 2 || opt.rates_W == 4) &&
        (Ns + opt.rates_W - 1) / opt.rates_W <= 32)
        W = opt.rates_W;
    // q buffer rows: what is left of a third (W=4) of the SM's shared memory after the (C,g) state
    const size_t state = sizeof(double) * 2 * 32 * (size_t)(Ns + 1) + sizeof(double) * 32 * 2 * W;
    const size_t per_block = (227 * 1024) / (W == 4 ? 3 : (W == 2 ? 6 : 12)) - 1024;
    int Rc = state + 32 * 256 <= per_block ? (int)((per_block - state) / 256) : 32;
    Rc = std::min(Rc, 128) / (2 * W) * (2 * W);  // whole pairs of reactions per warp
    Rc = std::max(Rc, 2 * W);
    o.W = W, o.Rc = Rc;

    const int16_t *reac = t->reac, *prod = t->prod;
    auto slot = [&](const int16_t *tab, int s, int r) { return (int)tab[(size_t)s * Nr + r]; };
    std::vector<int> order;
    std::vector<int4> chunks;
    for (int kind = 0; kind < 3; ++kind) {
        const int r0 = kind == 0 ? 0 : (kind == 1 ? Ne : Ne + N3), r1 = kind == 0 ? Ne : (kind == 1 ? Ne + N3 : Nr);
        for (int generic = 0; generic < 2; ++generic) {
            std::vector<int> grp;
            for (int r = r0; r < r1; ++r)
                if ((slot(reac, 2, r) >= 0 || slot(prod, 2, r) >= 0) == (generic == 1)) grp.push_back(r);
            for (size_t i = 0; i < grp.size(); i += Rc) {
                const int cnt = (int)std::min<size_t>(Rc, grp.size() - i);
                chunks.push_back(make_int4(kind | generic << 2, (int)order.size(), cnt, 0));
                order.insert(order.end(), grp.begin() + i, grp.begin() + i + cnt);
            }
        }
    }
    o.n_chunks = (int)chunks.size();

    const int row = 32 * 16;  // bytes per species row of the (C, g) state
    std::vector<double> rc((size_t)Nr * 4);
    std::vector<int> rs((size_t)Nr * 8);
    for (int i = 0; i < Nr; ++i) {
        const int r = order[i];
        int nf = 0, nbk = 0;
        for (int s = 0; s < 3; ++s) nf += slot(reac, s, r) >= 0, nbk += slot(prod, s, r) >= 0;
        rc[4 * (size_t)i + 0] = crf::kLog2e * t->lnA[r];
        rc[4 * (size_t)i + 1] = crf::kLog2e * t->beta[r];
        rc[4 * (size_t)i + 2] = -crf::kLog2e * t->Ea_R[r];
        rc[4 * (size_t)i + 3] = double(nbk - nf);
        auto off = [&](int k) { return (k >= 0 ? k : Ns) * row; };  // row Ns is the dummy species (C = 1, g = 0)
        int *q = rs.data() + 8 * (size_t)i;
        q[0] = off(slot(reac, 0, r)), q[1] = off(slot(reac, 1, r)), q[2] = off(slot(prod, 0, r)),
        q[3] = off(slot(prod, 1, r));
        q[4] = off(slot(reac, 2, r)), q[5] = off(slot(prod, 2, r));
        q[6] = r >= Ne ? r - Ne : 0;            // row of the efficiency CSR
        q[7] = r >= Ne + N3 ? r - Ne - N3 : 0;  // row of the falloff table
    }
    // incidence lists per chunk, species-major: omega_k += nu * q
    std::vector<int> inc_ptr;
    std::vector<double2> inc;
    for (const int4 &ch : chunks) {
        for (int k = 0; k < Ns; ++k) {
            inc_ptr.push_back((int)inc.size());
            for (int rl = 0; rl < ch.z; ++rl) {
                const int r = order[ch.y + rl];
                int nu = 0;
                for (int s = 0; s < 3; ++s) nu += (slot(prod, s, r) == k) - (slot(reac, s, r) == k);
                if (nu != 0) {
                    const int64_t bits = (int64_t)rl * 256;
                    double as_double;
                    std::memcpy(&as_double, &bits, sizeof(double));
                    inc.push_back(make_double2((double)nu, as_double));
                }
            }
        }
        inc_ptr.push_back((int)inc.size());
    }
    std::vector<double> troe((size_t)std::max(Nt, 1) * 8, 0.0);
    for (int i = 0; i < Nt; ++i) {
        double *q = troe.data() + 8 * (size_t)i;
        q[0] = crf::kLog2e * t->lnA0[i], q[1] = crf::kLog2e * t->beta0[i], q[2] = -crf::kLog2e * t->Ea0_R[i];
        q[3] = t->alpha[i], q[4] = -crf::kLog2e / t->T3[i], q[5] = -crf::kLog2e / t->T1[i], q[6] = -crf::kLog2e * t->T2[i];
    }
    // NASA sets: g/(RT) * log2(e) = c0 (1 - ln T) + T (c1 + T (c2 + T (c3 + T c4))) + c5/T + c6 ; h/(RT) plain
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
            if (rg == 1) g[7] = 1.0 / t->W[k];
        }
    o.chunk = b.add(chunks), o.rc = b.add(rc), o.rs = b.add(rs), o.inc_ptr = b.add(inc_ptr), o.inc = b.add(inc);
    o.troe = b.add(troe), o.gco = b.add(gco), o.hco = b.add(hco);
    return o;
}
