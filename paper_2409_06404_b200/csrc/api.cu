// api.cu -- the C ABI of libcrf.so (include/crf.h): mechanism construction (host re-layout of the
// packed tables + upload), argument checks, dispatch to the kernel launchers, the host-buffer
// pipeline crf_step_host and the FP64 probe.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/crf_diag.h"
#include "crf_internal.h"
#include "host_plan.h"
#include "launch.h"

namespace {

thread_local std::string g_err;
std::atomic<int64_t> g_launches{0};

int fail(int code, const std::string &msg)
{
    g_err = msg;
    return code;
}
int fail_cuda(cudaError_t e, const char *where)
{
    return fail(CRF_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
bool misaligned(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

constexpr int kSlots = 3;                       // pipeline depth of crf_step_host (four measured: no difference)
constexpr int64_t kPipeOutBytes = 128 << 20;    // output bytes of a chunk to aim for (64 MB, 256 MB measured: no difference)
constexpr int kStoich = 3;              // reactant / product slots of a reaction (crf_tables.reac, prod)
// points per chunk of crf_step_host: a power of two whose double-precision outputs, 8 (2 Ns + 5) bytes per point, come
// to about kPipeOutBytes per chunk (65536 points at 118 species, 524288 at 21 and fewer): copies long enough to run at the
// link's rate, enough chunks to overlap the two copy directions and the kernels
int64_t pipe_chunk_points(int Ns)
{
    int64_t c = 16384;
    while (c < (1 << 19) && 2 * c * 8 * (2 * (int64_t)Ns + 5) <= kPipeOutBytes + (kPipeOutBytes >> 1)) c *= 2;
    return c;
}

}  // namespace

void crf_count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

struct crf_mech {
    DevTables dev{};
    crf_plan_info info{};
    void *block = nullptr;
    cudaStream_t stream = nullptr;
    // crf_step_host resources (lazy)
    cudaStream_t pipe_stream[kSlots] = {};
    double *pipe_buf[kSlots] = {};
    int64_t pipe_chunk = 0;
};

extern "C" {

const char *crf_last_error(void) { return g_err.c_str(); }
int64_t crf_launch_count(void) { return g_launches.load(); }

}  // extern "C"

namespace {

int mech_create(const crf_tables *t, const crf_plan_options &opt, crf_mech **out)
{
    if (t->version != CRF_TABLES_VERSION) return fail(CRF_EINVAL, "crf_mech_create: tables version mismatch");
    const int Ns = t->Ns, Nr = t->Nr, N3 = t->N3, Nt = t->Nt;
    if (Ns < 1 || Nr < 0 || N3 < 0 || Nt < 0 || N3 + Nt > Nr) return fail(CRF_EINVAL, "crf_mech_create: bad counts");
    if (Ns > CRF_MAX_SPECIES) return fail(CRF_EUNSUPPORTED, "crf_mech_create: more than CRF_MAX_SPECIES (220) species");
    if (!(t->p_ref > 0.0)) return fail(CRF_EINVAL, "crf_mech_create: p_ref must be positive");
    const void *need[] = {t->W, t->Tmid, t->nasa_lo, t->nasa_hi, t->mu_c, t->lam_c, t->D_c};
    for (const void *q : need)
        if (!q) return fail(CRF_EINVAL, "crf_mech_create: null table");
    if (Nr > 0 && (!t->lnA || !t->beta || !t->Ea_R || !t->reac || !t->prod))
        return fail(CRF_EINVAL, "crf_mech_create: null reaction table");
    if (N3 + Nt > 0 && (!t->eff_ptr || !t->eff_idx || !t->eff_val))
        return fail(CRF_EINVAL, "crf_mech_create: null efficiency table");
    if (Nt > 0 && (!t->lnA0 || !t->beta0 || !t->Ea0_R || !t->alpha || !t->T3 || !t->T1 || !t->T2))
        return fail(CRF_EINVAL, "crf_mech_create: null falloff table");
    for (int k = 0; k < Ns; ++k)
        if (!(t->W[k] > 0.0)) return fail(CRF_EINVAL, "crf_mech_create: molar masses must be positive");

    // ---- derived host tables ----
    std::vector<double> W(t->W, t->W + Ns), rW(Ns), Tmid(t->Tmid, t->Tmid + Ns), wq(Ns);
    for (int k = 0; k < Ns; ++k) {
        rW[k] = 1.0 / W[k];
        wq[k] = 1.0 / std::sqrt(std::sqrt(W[k]));
    }
    std::vector<double> cpc(2 * 5 * Ns), hc(2 * 6 * Ns), gc(2 * 7 * Ns), sc(2 * 6 * Ns);
    for (int rg = 0; rg < 2; ++rg) {
        const double *a = rg == 0 ? t->nasa_lo : t->nasa_hi;  // [7][Ns]
        for (int k = 0; k < Ns; ++k) {
            const double a1 = a[0 * Ns + k], a2 = a[1 * Ns + k], a3 = a[2 * Ns + k], a4 = a[3 * Ns + k],
                         a5 = a[4 * Ns + k], a6 = a[5 * Ns + k], a7 = a[6 * Ns + k];
            double *c = cpc.data() + rg * 5 * Ns + k;
            c[0] = a1, c[Ns] = a2, c[2 * Ns] = a3, c[3 * Ns] = a4, c[4 * Ns] = a5;
            double *h = hc.data() + rg * 6 * Ns + k;
            h[0] = a1, h[Ns] = a2 / 2.0, h[2 * Ns] = a3 / 3.0, h[3 * Ns] = a4 / 4.0, h[4 * Ns] = a5 / 5.0,
            h[5 * Ns] = a6;
            double *s = sc.data() + rg * 6 * Ns + k;
            s[0] = a1, s[Ns] = a2, s[2 * Ns] = a3 / 2.0, s[3 * Ns] = a4 / 3.0, s[4 * Ns] = a5 / 4.0, s[5 * Ns] = a7;
            double *g = gc.data() + rg * 7 * Ns + k;
            g[0] = a1, g[Ns] = -a2 / 2.0, g[2 * Ns] = -a3 / 6.0, g[3 * Ns] = -a4 / 12.0, g[4 * Ns] = -a5 / 20.0,
            g[5 * Ns] = a6, g[6 * Ns] = -a7;
        }
    }
    std::vector<double> thermo_tab(14 * (size_t)Ns, 0.0);
    for (int k = 0; k < Ns; ++k) {
        for (int c = 0; c < 6; ++c) {
            thermo_tab[14 * (size_t)k + c] = t->nasa_lo[(size_t)c * Ns + k] / W[k];
            thermo_tab[14 * (size_t)k + 6 + c] = t->nasa_hi[(size_t)c * Ns + k] / W[k];
        }
        thermo_tab[14 * (size_t)k + 12] = Tmid[k];
    }
    std::vector<double> lnA(t->lnA, t->lnA + Nr), beta(t->beta, t->beta + Nr), Ea_R(t->Ea_R, t->Ea_R + Nr), dnu(Nr);
    std::vector<int16_t> reac(t->reac, t->reac + (size_t)kStoich * Nr), prod(t->prod, t->prod + (size_t)kStoich * Nr);
    for (int r = 0; r < Nr; ++r) {
        int nf = 0, nb = 0;
        for (int s = 0; s < kStoich; ++s) {
            const int a = reac[(size_t)s * Nr + r], b = prod[(size_t)s * Nr + r];
            if (a >= Ns || b >= Ns || a < -1 || b < -1)
                return fail(CRF_EINVAL, "crf_mech_create: species index out of range");
            nf += a >= 0;
            nb += b >= 0;
        }
        if (nf == 0 || nb == 0) return fail(CRF_EINVAL, "crf_mech_create: reaction without reactant or product");
        dnu[r] = double(nb - nf);
    }
    const int nM = N3 + Nt;
    std::vector<int32_t> eff_ptr(nM + 1, 0);
    std::vector<int16_t> eff_idx;
    std::vector<double> eff_val;
    if (nM > 0) {
        eff_ptr.assign(t->eff_ptr, t->eff_ptr + nM + 1);
        if (eff_ptr[0] != 0) return fail(CRF_EINVAL, "crf_mech_create: eff_ptr[0] must be 0");
        for (int r = 0; r < nM; ++r)
            if (eff_ptr[r + 1] < eff_ptr[r]) return fail(CRF_EINVAL, "crf_mech_create: eff_ptr not monotone");
        eff_idx.assign(t->eff_idx, t->eff_idx + eff_ptr[nM]);
        eff_val.assign(t->eff_val, t->eff_val + eff_ptr[nM]);
        for (int16_t k : eff_idx)
            if (k < 0 || k >= Ns) return fail(CRF_EINVAL, "crf_mech_create: efficiency species out of range");
    }
    std::vector<double> lnA0, beta0, Ea0_R, alpha, rT3, rT1, T2;
    if (Nt > 0) {
        lnA0.assign(t->lnA0, t->lnA0 + Nt);
        beta0.assign(t->beta0, t->beta0 + Nt);
        Ea0_R.assign(t->Ea0_R, t->Ea0_R + Nt);
        alpha.assign(t->alpha, t->alpha + Nt);
        T2.assign(t->T2, t->T2 + Nt);
        rT3.resize(Nt);
        rT1.resize(Nt);
        for (int i = 0; i < Nt; ++i) {
            // (T3 = 1e-30 and T1 = T2 = 1e30 or inf are the Chemkin way of switching a term off: accepted)
            if (!(t->T3[i] != 0.0) || !(t->T1[i] != 0.0) || std::isnan(t->T2[i]) || !std::isfinite(t->alpha[i]))
                return fail(CRF_EINVAL, "crf_mech_create: Troe parameters: T3 and T1 must be non-zero, alpha finite");
            rT3[i] = 1.0 / t->T3[i];
            rT1[i] = 1.0 / t->T1[i];
        }
    }
    const int npair = Ns * (Ns + 1) / 2;
    std::vector<double> mu_c(t->mu_c, t->mu_c + 4 * Ns), lam_c(t->lam_c, t->lam_c + 4 * Ns), nDc(4 * (size_t)npair),
        wilke(Ns * (size_t)Ns);
    for (int q = 0; q < npair; ++q)
        for (int c = 0; c < 4; ++c) nDc[4 * (size_t)q + c] = -t->D_c[(size_t)c * npair + q];
    for (int k = 0; k < Ns; ++k)
        for (int j = 0; j < Ns; ++j) wilke[(size_t)k * Ns + j] = 1.0 / std::sqrt(8.0 * (1.0 + W[k] / W[j]));

    // ---- one device block ----
    BlockBuilder b;
    const size_t oW = b.add(W), orW = b.add(rW), oTm = b.add(Tmid), ocp = b.add(cpc), ohc = b.add(hc), ogc = b.add(gc),
                 osc = b.add(sc), olnA = b.add(lnA), obeta = b.add(beta), oEa = b.add(Ea_R), odnu = b.add(dnu),
                 oreac = b.add(reac), oprod = b.add(prod), oep = b.add(eff_ptr), oei = b.add(eff_idx),
                 oev = b.add(eff_val), olnA0 = b.add(lnA0), ob0 = b.add(beta0), oE0 = b.add(Ea0_R), oal = b.add(alpha),
                 orT3 = b.add(rT3), orT1 = b.add(rT1), oT2 = b.add(T2), omu = b.add(mu_c), olam = b.add(lam_c),
                 onD = b.add(nDc), owk = b.add(wilke), owq = b.add(wq), otht = b.add(thermo_tab);
    const TransportPlanOffsets tpo = build_transport_plan(t, opt, b);
    const RatesPlanOffsets rpo = build_rates_plan(t, opt, b);
    const RatesSmemPlanOffsets rso = build_rates_smem_plan(t, opt, b);
    // (small mechanisms run the thread kernel for crf_production_rates; the warp-group plan is still built: it serves the
    // pair / difference-quotient / fused right-hand-side calls, which evaluate two states or emit by-products per launch)
    const RatesGroupPlanOffsets rgo = build_rates_group_plan(t, opt, b);
    // what will run, and whether that is what was asked for
    crf_plan_info info{};
    info.rates_kernel = rso.W > 0 ? CRF_RATES_THREAD
                                  : (rgo.W > 0 ? CRF_RATES_GROUP : (rpo.W > 0 ? CRF_RATES_STAGED : CRF_RATES_GENERIC));
    if (rso.W > 0)
        info.rates_W = rso.W, info.rates_PPL = rso.PPL, info.rates_Rc = rso.Rc, info.rates_chunks = rso.n_chunks,
        info.rates_stage_bytes = rso.stage_bytes, info.rates_tmem_cols = (opt.rates_tmem != 1 && 6 * (Ns + 1) <= 512) ? 6 * (Ns + 1) : 0;
    else if (rgo.W > 0)
        info.rates_W = rgo.W, info.rates_PPL = rgo.PPL, info.rates_Rc = rgo.Rc, info.rates_chunks = rgo.n_chunks,
        info.rates_stage_bytes = rgo.stage_bytes, info.rates_tmem_cols = rgo.tm_cols;
    else if (rpo.W > 0)
        info.rates_W = rpo.W, info.rates_PPL = 1, info.rates_Rc = rpo.Rc, info.rates_chunks = rpo.n_chunks;
    info.transport_kernel = tpo.W > 0 ? CRF_TRANSPORT_TILED : (tpo.small_n > 0 ? CRF_TRANSPORT_SMALL : CRF_TRANSPORT_GENERIC);
    if (tpo.W > 0)
        info.transport_W = tpo.W, info.transport_PPL = tpo.PPL, info.transport_nb = tpo.nbp, info.transport_TS = tpo.TS,
        info.transport_stage_blocks = tpo.n_wilke + tpo.n_rounds, info.transport_stage_bytes = tpo.stage_bytes;
    info.thermo_sets = opt.thermo_sets == 1 ? 1 : 2;
    if (opt.rates_kernel != CRF_RATES_AUTO && opt.rates_kernel != info.rates_kernel && Nr > 0)
        return fail(CRF_EUNSUPPORTED, "crf_mech_create_ex: the requested rates kernel does not admit this mechanism");
    if (opt.transport_kernel != CRF_TRANSPORT_AUTO && opt.transport_kernel != info.transport_kernel)
        return fail(CRF_EUNSUPPORTED, "crf_mech_create_ex: the requested transport kernel does not admit this mechanism");
    crf_mech *mech = new (std::nothrow) crf_mech;
    if (!mech) return fail(CRF_ECUDA, "crf_mech_create: out of host memory");
    cudaError_t e = cudaMalloc(&mech->block, b.bytes.size());
    if (e != cudaSuccess) {
        delete mech;
        return fail_cuda(e, "crf_mech_create: cudaMalloc");
    }
    e = cudaMemcpy(mech->block, b.bytes.data(), b.bytes.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaFree(mech->block);
        delete mech;
        return fail_cuda(e, "crf_mech_create: cudaMemcpy");
    }
    const unsigned char *base = static_cast<const unsigned char *>(mech->block);
    auto D = [&](size_t off) { return reinterpret_cast<const double *>(base + off); };
    DevTables &d = mech->dev;
    d.Ns = Ns, d.Nr = Nr, d.Ne = Nr - N3 - Nt, d.N3 = N3, d.Nt = Nt, d.npair = npair, d.p_ref = t->p_ref;
    d.W = D(oW), d.rW = D(orW), d.Tmid = D(oTm), d.cpc = D(ocp), d.hc = D(ohc), d.gc = D(ogc), d.sc = D(osc);
    d.lnA = D(olnA), d.beta = D(obeta), d.Ea_R = D(oEa), d.dnu = D(odnu);
    d.reac = reinterpret_cast<const int16_t *>(base + oreac);
    d.prod = reinterpret_cast<const int16_t *>(base + oprod);
    d.eff_ptr = reinterpret_cast<const int32_t *>(base + oep);
    d.eff_idx = reinterpret_cast<const int16_t *>(base + oei);
    d.eff_val = D(oev);
    d.lnA0 = D(olnA0), d.beta0 = D(ob0), d.Ea0_R = D(oE0), d.alpha = D(oal), d.rT3 = D(orT3), d.rT1 = D(orT1),
    d.T2 = D(oT2);
    d.thermo_tab = D(otht);
    d.thermo_sets = opt.thermo_sets == 1 ? 1 : 2;
    d.mu_c = D(omu), d.lam_c = D(olam), d.nDc = D(onD), d.wilke_c = D(owk), d.wq = D(owq);
    TransportPlan &tp = d.tp;
    tp.W = tpo.W, tp.PPL = tpo.PPL, tp.NsP = tpo.NsP, tp.nb = tpo.nb, tp.n_wilke = tpo.n_wilke, tp.n_rounds = tpo.n_rounds;
    tp.TS = tpo.TS;
    tp.stage_bytes = tpo.stage_bytes;
    tp.small = D(tpo.small), tp.small_n = tpo.small_n;
    tp.rounds = reinterpret_cast<const int4 *>(base + tpo.rounds);
    tp.pair_coef = base + tpo.pair_coef, tp.wilke_cP = D(tpo.wilke_cP), tp.sp = D(tpo.sp), tp.Ddiag = D(tpo.Ddiag);
    RatesPlan &rp = d.rp;
    rp.W = rpo.W, rp.Rc = rpo.Rc, rp.n_chunks = rpo.n_chunks;
    rp.chunk = reinterpret_cast<const int4 *>(base + rpo.chunk);
    rp.rc = D(rpo.rc);
    rp.rs = reinterpret_cast<const int4 *>(base + rpo.rs);
    rp.inc_ptr = reinterpret_cast<const int *>(base + rpo.inc_ptr);
    rp.inc = reinterpret_cast<const double2 *>(base + rpo.inc);
    rp.troe = D(rpo.troe), rp.gco = D(rpo.gco), rp.hco = D(rpo.hco);
    RatesSmemPlan &rs = d.rs;
    rs.tmem = (opt.rates_tmem != 1 && 6 * (Ns + 1) <= 512) ? 1 : 0;
    rs.W = rso.W, rs.PPL = rso.PPL, rs.maxown = rso.maxown, rs.Rc = rso.Rc, rs.n_chunks = rso.n_chunks, rs.stage_bytes = rso.stage_bytes;
    rs.chunk = reinterpret_cast<const int4 *>(base + rso.chunk);
    rs.stage = base + rso.stage;
    rs.gco = D(rso.gco), rs.hco = D(rso.hco);
    RatesGroupPlan &rg = d.rg;
    rg.W = rgo.W, rg.PPL = rgo.PPL, rg.maxown = rgo.maxown, rg.Rc = rgo.Rc, rg.n_chunks = rgo.n_chunks,
    rg.stage_bytes = rgo.stage_bytes, rg.q_rows = rgo.q_rows, rg.tm_cols = rgo.tm_cols, rg.log2_c0 = rgo.log2_c0;
    rg.chunk = reinterpret_cast<const int4 *>(base + rgo.chunk);
    rg.stage = base + rgo.stage;
    rg.gco = D(rgo.gco), rg.hco = D(rgo.hco);
    rg.own = reinterpret_cast<const int *>(base + rgo.own);
    info.rates_smem_bytes = (int)rates_dynamic_smem(d);
    info.transport_smem_bytes = (int)transport_dynamic_smem(d);
    mech->info = info;
    *out = mech;
    return CRF_OK;
}

}  // namespace

extern "C" {

int crf_mech_create_ex(const crf_tables *t, const crf_plan_options *options, crf_mech **out)
{
    if (!t || !out) return fail(CRF_EINVAL, "crf_mech_create: null argument");
    crf_plan_options opt{};
    if (options) opt = *options;
    for (int32_t r : opt.reserved)
        if (r != 0) return fail(CRF_EINVAL, "crf_mech_create_ex: reserved option fields must be 0");
    if (opt.transport_TS != 0 && opt.transport_TS != 7 && opt.transport_TS != 8)
        return fail(CRF_EINVAL, "crf_mech_create_ex: transport_TS must be 0, 7 or 8");
    if (opt.thermo_sets < 0 || opt.thermo_sets > 2) return fail(CRF_EINVAL, "crf_mech_create_ex: thermo_sets must be 0, 1 or 2");
    try {  // the host re-layout allocates: no C++ exception may cross the boundary
        return mech_create(t, opt, out);
    } catch (const std::bad_alloc &) {
        return fail(CRF_ECUDA, "crf_mech_create: out of host memory");
    } catch (const std::exception &e) {
        return fail(CRF_EINVAL, std::string("crf_mech_create: ") + e.what());
    } catch (...) {
        return fail(CRF_EINVAL, "crf_mech_create: unexpected exception");
    }
}

int crf_mech_create(const crf_tables *t, crf_mech **out) { return crf_mech_create_ex(t, nullptr, out); }

int crf_mech_plan_info(const crf_mech *mech, crf_plan_info *info)
{
    if (!mech || !info) return fail(CRF_EINVAL, "crf_mech_plan_info: null argument");
    *info = mech->info;
    return CRF_OK;
}

void crf_mech_destroy(crf_mech *mech)
{
    if (!mech) return;
    for (int s = 0; s < kSlots; ++s) {
        if (mech->pipe_buf[s]) cudaFree(mech->pipe_buf[s]);
        if (mech->pipe_stream[s]) cudaStreamDestroy(mech->pipe_stream[s]);
    }
    if (mech->block) cudaFree(mech->block);
    delete mech;
}

int crf_mech_set_stream(crf_mech *mech, void *cuda_stream)
{
    if (!mech) return fail(CRF_EINVAL, "crf_mech_set_stream: null mechanism");
    mech->stream = static_cast<cudaStream_t>(cuda_stream);
    return CRF_OK;
}
int crf_mech_num_species(const crf_mech *mech) { return mech ? mech->dev.Ns : CRF_EINVAL; }
int crf_mech_num_reactions(const crf_mech *mech) { return mech ? mech->dev.Nr : CRF_EINVAL; }

#define CRF_CHECK_COMMON(name)                                                  \
    if (!mech) return fail(CRF_EINVAL, name ": null mechanism");                \
    if (n < 0) return fail(CRF_EINVAL, name ": negative n");                    \
    if (n == 0) return CRF_OK;                                                  \
    if (n > (int64_t)2147483647 * 32) return fail(CRF_EINVAL, name ": n too large");

int crf_thermo(const crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n, double *cp,
               double *h)
{
    CRF_CHECK_COMMON("crf_thermo")
    if (!T || !Y || !cp || !h) return fail(CRF_EINVAL, "crf_thermo: null pointer");
    if (misaligned(T) || misaligned(Y) || misaligned(cp) || misaligned(h) || misaligned(p))
        return fail(CRF_EINVAL, "crf_thermo: pointers must be 16-byte aligned");
    cudaError_t e = launch_thermo(mech->dev, T, Y, n, cp, h, mech->stream);
    return e == cudaSuccess ? CRF_OK : fail_cuda(e, "crf_thermo");
}

int crf_thermo_species(const crf_mech *mech, const double *T, int64_t n, double *cpk, double *hk, double *sk)
{
    CRF_CHECK_COMMON("crf_thermo_species")
    if (!T) return fail(CRF_EINVAL, "crf_thermo_species: null pointer");
    if (misaligned(T) || misaligned(cpk) || misaligned(hk) || misaligned(sk))
        return fail(CRF_EINVAL, "crf_thermo_species: pointers must be 16-byte aligned");
    cudaError_t e = launch_thermo_species(mech->dev, T, n, cpk, hk, sk, mech->stream);
    return e == cudaSuccess ? CRF_OK : fail_cuda(e, "crf_thermo_species");
}

int crf_production_rates(const crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n,
                         double *omega, double *qdot)
{
    CRF_CHECK_COMMON("crf_production_rates")
    if (!T || !p || !Y || !omega || !qdot) return fail(CRF_EINVAL, "crf_production_rates: null pointer");
    if (misaligned(T) || misaligned(p) || misaligned(Y) || misaligned(omega) || misaligned(qdot))
        return fail(CRF_EINVAL, "crf_production_rates: pointers must be 16-byte aligned");
    cudaError_t e = launch_rates(mech->dev, T, p, Y, n, omega, qdot, mech->stream);
    return e == cudaSuccess ? CRF_OK : fail_cuda(e, "crf_production_rates");
}

int crf_mix_transport(const crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n, double *mu,
                      double *lambda, double *rhoD)
{
    CRF_CHECK_COMMON("crf_mix_transport")
    if (!T || !Y || !mu || !lambda || !rhoD) return fail(CRF_EINVAL, "crf_mix_transport: null pointer");
    if (misaligned(T) || misaligned(p) || misaligned(Y) || misaligned(mu) || misaligned(lambda) || misaligned(rhoD))
        return fail(CRF_EINVAL, "crf_mix_transport: pointers must be 16-byte aligned");
    cudaError_t e = launch_transport(mech->dev, T, p, Y, n, mu, lambda, rhoD, mech->stream);
    return e == cudaSuccess ? CRF_OK : fail_cuda(e, "crf_mix_transport");
}

int crf_production_rates_pair(const crf_mech *mech, const double *T, const double *p, const double *Y, const double *T2,
                              const double *p2, const double *Y2, int64_t n, double *omega, double *qdot, double *omega2,
                              double *qdot2)
{
    CRF_CHECK_COMMON("crf_production_rates_pair")
    if (!T || !p || !Y || !T2 || !p2 || !Y2 || !omega || !qdot || !omega2 || !qdot2)
        return fail(CRF_EINVAL, "crf_production_rates_pair: null pointer");
    for (const void *q : {(const void *)T, (const void *)p, (const void *)Y, (const void *)T2, (const void *)p2,
                          (const void *)Y2, (const void *)omega, (const void *)qdot, (const void *)omega2, (const void *)qdot2})
        if (misaligned(q)) return fail(CRF_EINVAL, "crf_production_rates_pair: pointers must be 16-byte aligned");
    cudaError_t e;
    RatesIO io = rates_io(T, p, Y, omega, qdot);
    io.T2 = T2, io.p2 = p2, io.Y2 = Y2, io.omega2 = omega2, io.qdot2 = qdot2, io.mode = 1;
    if (rates_thread_tm_serves(mech->dev, io)) {  // (small mechanisms: the thread kernel evaluates both states per launch)
        e = launch_rates_thread_io(mech->dev, io, n, mech->stream);
    } else if (mech->dev.rg.W > 0 && mech->dev.rg.PPL == 2) {
        e = launch_rates_group(mech->dev, io, n, mech->stream);
    } else {  // no plan that shares a launch: two launches of whatever kernel the mechanism runs
        e = launch_rates(mech->dev, T, p, Y, n, omega, qdot, mech->stream);
        if (e == cudaSuccess) e = launch_rates(mech->dev, T2, p2, Y2, n, omega2, qdot2, mech->stream);
    }
    return e == cudaSuccess ? CRF_OK : fail_cuda(e, "crf_production_rates_pair");
}

int crf_production_rates_jv(const crf_mech *mech, const double *T, const double *p, const double *Y, const double *dT,
                            const double *dp, const double *dY, double sigma, int64_t n, double *omega, double *qdot,
                            double *Jomega, double *Jqdot)
{
    CRF_CHECK_COMMON("crf_production_rates_jv")
    if (!T || !p || !Y || !dT || !dY || !Jomega || !Jqdot) return fail(CRF_EINVAL, "crf_production_rates_jv: null pointer");
    if (!(sigma != 0.0) || !std::isfinite(sigma)) return fail(CRF_EINVAL, "crf_production_rates_jv: sigma must be finite and non-zero");
    if ((omega == nullptr) != (qdot == nullptr))
        return fail(CRF_EINVAL, "crf_production_rates_jv: omega and qdot must be given or omitted together");
    for (const void *q : {(const void *)T, (const void *)p, (const void *)Y, (const void *)dT, (const void *)dp,
                          (const void *)dY, (const void *)omega, (const void *)qdot, (const void *)Jomega, (const void *)Jqdot})
        if (misaligned(q)) return fail(CRF_EINVAL, "crf_production_rates_jv: pointers must be 16-byte aligned");
    RatesIO io = rates_io(T, p, Y, omega, qdot);
    io.T2 = dT, io.Y2 = dY, io.omega2 = Jomega, io.qdot2 = Jqdot, io.sigma = sigma, io.inv_sigma = 1.0 / sigma, io.mode = 2;
    io.p2 = dp ? dp : p, io.sigma_p = dp ? sigma : 0.0;  // (no pressure perturbation: p + 0 p)
    cudaError_t e;
    if (rates_thread_tm_serves(mech->dev, io))
        e = launch_rates_thread_io(mech->dev, io, n, mech->stream);
    else if (mech->dev.rg.W > 0 && mech->dev.rg.PPL == 2)
        e = launch_rates_group(mech->dev, io, n, mech->stream);
    else
        return fail(CRF_EUNSUPPORTED, "crf_production_rates_jv: this mechanism has no warp-group plan with two states per lane "
                                      "(use crf_production_rates_pair on a perturbed copy)");
    return e == cudaSuccess ? CRF_OK : fail_cuda(e, "crf_production_rates_jv");
}

int crf_production_rates_jv_base(const crf_mech *mech, const double *T, const double *p, const double *Y, const double *dT,
                                 const double *dp, const double *dY, double sigma, int64_t n, const double *omega,
                                 const double *qdot, double *Jomega, double *Jqdot)
{
    CRF_CHECK_COMMON("crf_production_rates_jv_base")
    if (!T || !p || !Y || !dT || !dY || !omega || !qdot || !Jomega || !Jqdot)
        return fail(CRF_EINVAL, "crf_production_rates_jv_base: null pointer");
    if (!(sigma != 0.0) || !std::isfinite(sigma))
        return fail(CRF_EINVAL, "crf_production_rates_jv_base: sigma must be finite and non-zero");
    for (const void *q : {(const void *)T, (const void *)p, (const void *)Y, (const void *)dT, (const void *)dp,
                          (const void *)dY, (const void *)omega, (const void *)qdot, (const void *)Jomega, (const void *)Jqdot})
        if (misaligned(q)) return fail(CRF_EINVAL, "crf_production_rates_jv_base: pointers must be 16-byte aligned");
    // (the kernels read the base values through the output slots of RatesIO and do not write them in this mode)
    RatesIO io = rates_io(T, p, Y, const_cast<double *>(omega), const_cast<double *>(qdot));
    io.T2 = dT, io.Y2 = dY, io.omega2 = Jomega, io.qdot2 = Jqdot, io.sigma = sigma, io.inv_sigma = 1.0 / sigma, io.mode = 4;
    io.p2 = dp ? dp : p, io.sigma_p = dp ? sigma : 0.0;
    cudaError_t e;
    if (rates_thread_tm_serves(mech->dev, io))
        e = launch_rates_thread_io(mech->dev, io, n, mech->stream);
    else if (mech->dev.rg.W > 0)
        e = launch_rates_group(mech->dev, io, n, mech->stream);
    else
        return fail(CRF_EUNSUPPORTED, "crf_production_rates_jv_base: this mechanism runs a fall-back kernel (use "
                                      "crf_production_rates on a perturbed copy)");
    return e == cudaSuccess ? CRF_OK : fail_cuda(e, "crf_production_rates_jv_base");
}

int crf_rhs_pointwise(const crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n, double *omega,
                      double *qdot, double *cp, double *h, double *cpk, double *rho, double *Wbar, double *mu,
                      double *lambda, double *rhoD)
{
    CRF_CHECK_COMMON("crf_rhs_pointwise")
    if (!T || !p || !Y || !omega || !qdot || !cp || !h || !rho || !Wbar || !mu || !lambda || !rhoD)
        return fail(CRF_EINVAL, "crf_rhs_pointwise: null pointer (only cpk may be omitted)");
    for (const void *q : {(const void *)T, (const void *)p, (const void *)Y, (const void *)omega, (const void *)qdot,
                          (const void *)cp, (const void *)h, (const void *)cpk, (const void *)rho, (const void *)Wbar,
                          (const void *)mu, (const void *)lambda, (const void *)rhoD})
        if (misaligned(q)) return fail(CRF_EINVAL, "crf_rhs_pointwise: pointers must be 16-byte aligned");
    const DevTables &d = mech->dev;
    cudaStream_t st = mech->stream;
    cudaError_t e;
    RatesIO io = rates_io(T, p, Y, omega, qdot);
    io.cp = cp, io.h = h, io.cpk = cpk, io.rho = rho, io.Wbar = Wbar;
    if (rates_thread_tm_serves(d, io)) {
        e = launch_rates_thread_io(d, io, n, st);
    } else if (d.rg.W > 0) {
        // the thermodynamic by-products leave the production-rates kernel (it evaluates the NASA sets and the
        // composition anyway): no separate thermo pass, Y is read by two kernels instead of three
        e = launch_rates_group(d, io, n, st);
    } else {
        e = launch_rates(d, T, p, Y, n, omega, qdot, st);
        if (e == cudaSuccess) e = launch_thermo(d, T, Y, n, cp, h, st);
        if (e == cudaSuccess && cpk) e = launch_thermo_species(d, T, n, cpk, nullptr, nullptr, st);
        if (e == cudaSuccess) e = launch_density(d, T, p, Y, n, rho, Wbar, st);
    }
    if (e == cudaSuccess) e = launch_transport(d, T, p, Y, n, mu, lambda, rhoD, st);
    return e == cudaSuccess ? CRF_OK : fail_cuda(e, "crf_rhs_pointwise");
}

int crf_sem_diffusion(const crf_mech *mech, const double *h3, const double *T, const double *Wbar, const double *Y,
                      const double *lambda, const double *rhoD, int64_t nel, double *dY, double *dT)
{
    if (!mech) return fail(CRF_EINVAL, "crf_sem_diffusion: null mechanism");
    if (nel < 0) return fail(CRF_EINVAL, "crf_sem_diffusion: negative element count");
    if (nel == 0) return CRF_OK;
    if (nel > (int64_t)1 << 31) return fail(CRF_EINVAL, "crf_sem_diffusion: too many elements");
    if (!h3 || !T || !Wbar || !Y || !lambda || !rhoD || !dY || !dT) return fail(CRF_EINVAL, "crf_sem_diffusion: null pointer");
    for (const void *q : {(const void *)h3, (const void *)T, (const void *)Wbar, (const void *)Y, (const void *)lambda,
                          (const void *)rhoD, (const void *)dY, (const void *)dT})
        if (misaligned(q)) return fail(CRF_EINVAL, "crf_sem_diffusion: pointers must be 16-byte aligned");
    cudaError_t e = launch_sem_diffusion(mech->dev, h3, T, Wbar, Y, lambda, rhoD, nel, dY, dT, mech->stream);
    return e == cudaSuccess ? CRF_OK : fail_cuda(e, "crf_sem_diffusion");
}

// Chunked host pipeline: slot s owns a stream and one device buffer holding, for a chunk of c points,
// T, p, Y[Ns], cp, h, qdot, mu, lambda, omega[Ns], rhoD[Ns] (each row c doubles), then the same output rows as floats
// (the single-precision staging of crf_step_host_f32).
}  // extern "C"

namespace {

template <class Out>
int step_host(const char *name, crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n, Out *cp, Out *h,
              Out *omega, Out *qdot, Out *mu, Out *lambda, Out *rhoD)
{
    constexpr bool kF32 = sizeof(Out) == 4;
    if (!mech) return fail(CRF_EINVAL, std::string(name) + ": null mechanism");
    if (n < 0) return fail(CRF_EINVAL, std::string(name) + ": negative n");
    if (n == 0) return CRF_OK;
    if (!T || !p || !Y) return fail(CRF_EINVAL, std::string(name) + ": null input pointer");
    // outputs are wanted per call: (cp, h), (omega, qdot), (mu, lambda, rhoD); a group that is NULL is neither computed nor copied
    const bool want_th = cp || h, want_ra = omega || qdot, want_tr = mu || lambda || rhoD;
    if ((want_th && (!cp || !h)) || (want_ra && (!omega || !qdot)) || (want_tr && (!mu || !lambda || !rhoD)))
        return fail(CRF_EINVAL, std::string(name) + ": the outputs of a call must be given together or all be NULL");
    if (!want_th && !want_ra && !want_tr) return fail(CRF_EINVAL, std::string(name) + ": no output requested");
    const int Ns = mech->dev.Ns;
    // (a call smaller than a chunk sizes the staging buffers for itself; a later, larger call allocates them again)
    const int64_t chunk = std::min(pipe_chunk_points(Ns), (n + 16383) / 16384 * 16384);
    const size_t rows = 7 + 3 * (size_t)Ns, out_rows = 5 + 2 * (size_t)Ns;
    cudaError_t e;
#define CRF_TRY(call)                                              \
    if ((e = (call)) != cudaSuccess) return fail_cuda(e, (std::string(name) + ": " #call).c_str());
    if (mech->pipe_chunk != chunk) {
        for (int s = 0; s < kSlots; ++s) {
            if (!mech->pipe_stream[s]) CRF_TRY(cudaStreamCreateWithFlags(&mech->pipe_stream[s], cudaStreamNonBlocking))
            if (mech->pipe_buf[s]) cudaFree(mech->pipe_buf[s]);
            mech->pipe_buf[s] = nullptr;  // (a failed cudaMalloc below must not leave a dangling pointer for crf_mech_destroy)
            e = cudaMalloc(&mech->pipe_buf[s], rows * chunk * sizeof(double) + out_rows * chunk * sizeof(float));
            if (e != cudaSuccess) {
                mech->pipe_buf[s] = nullptr;
                return fail_cuda(e, (std::string(name) + ": cudaMalloc").c_str());
            }
        }
        mech->pipe_chunk = chunk;
    }
    int slot = 0;
    for (int64_t off = 0; off < n; off += chunk, slot = (slot + 1) % kSlots) {
        const int64_t c = std::min(chunk, n - off);
        cudaStream_t st = mech->pipe_stream[slot];
        double *b = mech->pipe_buf[slot];
        double *dT = b, *dp = b + chunk, *dY = b + 2 * chunk, *dcp = dY + (size_t)Ns * chunk, *dh = dcp + chunk,
               *dq = dh + chunk, *dmu = dq + chunk, *dlam = dmu + chunk, *dom = dlam + chunk,
               *drD = dom + (size_t)Ns * chunk;
        float *f = reinterpret_cast<float *>(b + rows * chunk);  // the float image of the rows from dcp on, same order
        const size_t w = (size_t)c * sizeof(double);
        CRF_TRY(cudaMemcpyAsync(dT, T + off, w, cudaMemcpyHostToDevice, st))
        CRF_TRY(cudaMemcpyAsync(dp, p + off, w, cudaMemcpyHostToDevice, st))
        CRF_TRY(cudaMemcpy2DAsync(dY, w, Y + off, (size_t)n * sizeof(double), w, Ns, cudaMemcpyHostToDevice, st))
        // one output block of `nrow` rows (leading dimension c on the device, n on the host) back to the host, as doubles or,
        // rounded once on the device (round32, all blocks before the first copy), as floats
        auto round32 = [&](double *dev, int nrow) -> cudaError_t {
            return kF32 ? launch_f64_to_f32(dev, f + (dev - dcp), (int64_t)nrow * c, st) : cudaSuccess;
        };
        auto back = [&](Out *host, double *dev, int nrow) -> cudaError_t {
            if (!kF32)
                return cudaMemcpy2DAsync(host + off, (size_t)n * sizeof(Out), dev, w, w, nrow, cudaMemcpyDeviceToHost, st);
            float *fs = f + (dev - dcp);  // (rows are c doubles apart on the device: the float image keeps the same indices)
            return cudaMemcpy2DAsync(host + off, (size_t)n * sizeof(Out), fs, (size_t)c * sizeof(float), (size_t)c * sizeof(float),
                                     nrow, cudaMemcpyDeviceToHost, st);
        };
        // kernels see a compact chunk: leading dimension c.  All kernels of the chunk first, then all its copies back: a copy
        // between two kernels would hold the next kernel back (stream order) while the device-to-host engine, which takes
        // the copies of all slots in issue order, waits for that kernel behind it: the engine idled a third of the time
        // (C5 end to end 103-111 ms per step; with the copies behind the kernels it streams without gaps)
        if (want_th) CRF_TRY(launch_thermo(mech->dev, dT, dY, c, dcp, dh, st))
        if (want_ra) CRF_TRY(launch_rates(mech->dev, dT, dp, dY, c, dom, dq, st))
        if (want_tr) CRF_TRY(launch_transport(mech->dev, dT, dp, dY, c, dmu, dlam, drD, st))
        if (kF32) {
            if (want_th) {
                CRF_TRY(round32(dcp, 1))
                CRF_TRY(round32(dh, 1))
            }
            if (want_ra) {
                CRF_TRY(round32(dq, 1))
                CRF_TRY(round32(dom, Ns))
            }
            if (want_tr) {
                CRF_TRY(round32(dmu, 1))
                CRF_TRY(round32(dlam, 1))
                CRF_TRY(round32(drD, Ns))
            }
        }
        if (want_th) {
            CRF_TRY(back(cp, dcp, 1))
            CRF_TRY(back(h, dh, 1))
        }
        if (want_ra) {
            CRF_TRY(back(qdot, dq, 1))
            CRF_TRY(back(omega, dom, Ns))
        }
        if (want_tr) {
            CRF_TRY(back(mu, dmu, 1))
            CRF_TRY(back(lambda, dlam, 1))
            CRF_TRY(back(rhoD, drD, Ns))
        }
    }
    for (int s = 0; s < kSlots; ++s) CRF_TRY(cudaStreamSynchronize(mech->pipe_stream[s]))
#undef CRF_TRY
    return CRF_OK;
}

}  // namespace

extern "C" {

int crf_step_host(crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n, double *cp, double *h,
                  double *omega, double *qdot, double *mu, double *lambda, double *rhoD)
{
    return step_host<double>("crf_step_host", mech, T, p, Y, n, cp, h, omega, qdot, mu, lambda, rhoD);
}

int crf_step_host_f32(crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n, float *cp, float *h,
                      float *omega, float *qdot, float *mu, float *lambda, float *rhoD)
{
    return step_host<float>("crf_step_host_f32", mech, T, p, Y, n, cp, h, omega, qdot, mu, lambda, rhoD);
}

int crf_fp64_probe(int iters, double *inst_per_s)
{
    if (iters < 1 || !inst_per_s) return fail(CRF_EINVAL, "crf_fp64_probe: bad argument");
    cudaError_t e = launch_fp64_probe(iters, inst_per_s);
    return e == cudaSuccess ? CRF_OK : fail_cuda(e, "crf_fp64_probe");
}

}  // extern "C"

// ---- crf_step_host_static: crf_step_host for callers that may not allocate ----------------------------------------
// The device staging of the host-buffer call (inputs T, p, Y and the seven outputs of one batch) lives in a file-scope
// device array instead of the cudaMalloc'ed pipeline buffers of crf_step_host: 16 MiB that every GPU which loads
// libcrf.so holds until the process exits.  The call uses the mechanism's stream (crf_mech_set_stream), creates no
// stream and calls no cudaMalloc / cudaFree; its only set-up is the address lookup of the array, once per device.
// Every call on a device shares the array (also calls of different mechanisms): calls that overlap on the GPU race.
// No part of the array has to start at zero (every row a call reads was written by the same call before), so nothing
// is cleared; the array keeps the last call's contents.
namespace {

constexpr size_t kStaticDoubles = (size_t)2 << 20;  // 2 Mi doubles = 16 MiB
static __device__ __align__(256) double g_static_scratch[kStaticDoubles];

std::mutex g_static_mu;
double *g_static_ptr[64] = {};  // the DEVICE address of g_static_scratch on each device (the name itself is a host-side stand-in)

// blocks of the scratch start at multiples of 32 doubles (256 bytes)
size_t pad32(size_t v) { return (v + 31) & ~(size_t)31; }
size_t static_doubles(int Ns, int64_t n) { return 7 * pad32((size_t)n) + 3 * pad32((size_t)Ns * (size_t)n); }

}  // namespace

extern "C" {

int64_t crf_step_host_static_max_points(const crf_mech *mech)
{
    if (!mech) return fail(CRF_EINVAL, "crf_step_host_static_max_points: null mechanism");
    int64_t lo = 0, hi = (int64_t)kStaticDoubles;  // the largest n with static_doubles(Ns, n) <= kStaticDoubles
    while (lo < hi) {
        const int64_t mid = (lo + hi + 1) / 2;
        if (static_doubles(mech->dev.Ns, mid) <= kStaticDoubles)
            lo = mid;
        else
            hi = mid - 1;
    }
    return lo;
}

int crf_step_host_static(crf_mech *mech, const double *T, const double *p, const double *Y, int64_t n, double *cp, double *h,
                         double *omega, double *qdot, double *mu, double *lambda, double *rhoD)
{
    const char *name = "crf_step_host_static";
    if (!mech) return fail(CRF_EINVAL, std::string(name) + ": null mechanism");
    if (n < 0) return fail(CRF_EINVAL, std::string(name) + ": negative n");
    if (n == 0) return CRF_OK;
    if (!T || !p || !Y) return fail(CRF_EINVAL, std::string(name) + ": null input pointer");
    const bool want_th = cp || h, want_ra = omega || qdot, want_tr = mu || lambda || rhoD;
    if ((want_th && (!cp || !h)) || (want_ra && (!omega || !qdot)) || (want_tr && (!mu || !lambda || !rhoD)))
        return fail(CRF_EINVAL, std::string(name) + ": the outputs of a call must be given together or all be NULL");
    if (!want_th && !want_ra && !want_tr) return fail(CRF_EINVAL, std::string(name) + ": no output requested");
    const int Ns = mech->dev.Ns;
    if (n > (int64_t)kStaticDoubles || static_doubles(Ns, n) > kStaticDoubles)
        return fail(CRF_EINVAL, std::string(name) + ": n = " + std::to_string(n) + " points of " + std::to_string(Ns) +
                                    " species exceed the 16 MiB static scratch (at most " +
                                    std::to_string(crf_step_host_static_max_points(mech)) +
                                    " points per call for this mechanism; use crf_step_host, which allocates)");
    cudaError_t e;
#define CRF_TRY(call)                                              \
    if ((e = (call)) != cudaSuccess) return fail_cuda(e, (std::string(name) + ": " #call).c_str());
    int dev = 0;
    CRF_TRY(cudaGetDevice(&dev))
    if (dev < 0 || dev >= 64) return fail(CRF_EINVAL, std::string(name) + ": device ordinal out of range");
    double *b = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_static_mu);
        if (!g_static_ptr[dev]) {
            void *q = nullptr;
            CRF_TRY(cudaGetSymbolAddress(&q, g_static_scratch))
            g_static_ptr[dev] = static_cast<double *>(q);
        }
        b = g_static_ptr[dev];
    }
    cudaStream_t st = mech->stream;
    const size_t r1 = pad32((size_t)n), rN = pad32((size_t)Ns * (size_t)n);
    double *dT = b, *dp = dT + r1, *dY = dp + r1, *dcp = dY + rN, *dh = dcp + r1, *dq = dh + r1, *dmu = dq + r1, *dlam = dmu + r1,
           *dom = dlam + r1, *drD = dom + rN;
    const size_t w = (size_t)n * sizeof(double);
    CRF_TRY(cudaMemcpyAsync(dT, T, w, cudaMemcpyHostToDevice, st))
    CRF_TRY(cudaMemcpyAsync(dp, p, w, cudaMemcpyHostToDevice, st))
    CRF_TRY(cudaMemcpyAsync(dY, Y, w * Ns, cudaMemcpyHostToDevice, st))
    if (want_th) {
        CRF_TRY(launch_thermo(mech->dev, dT, dY, n, dcp, dh, st))
        CRF_TRY(cudaMemcpyAsync(cp, dcp, w, cudaMemcpyDeviceToHost, st))
        CRF_TRY(cudaMemcpyAsync(h, dh, w, cudaMemcpyDeviceToHost, st))
    }
    if (want_ra) {
        CRF_TRY(launch_rates(mech->dev, dT, dp, dY, n, dom, dq, st))
        CRF_TRY(cudaMemcpyAsync(qdot, dq, w, cudaMemcpyDeviceToHost, st))
        CRF_TRY(cudaMemcpyAsync(omega, dom, w * Ns, cudaMemcpyDeviceToHost, st))
    }
    if (want_tr) {
        CRF_TRY(launch_transport(mech->dev, dT, dp, dY, n, dmu, dlam, drD, st))
        CRF_TRY(cudaMemcpyAsync(mu, dmu, w, cudaMemcpyDeviceToHost, st))
        CRF_TRY(cudaMemcpyAsync(lambda, dlam, w, cudaMemcpyDeviceToHost, st))
        CRF_TRY(cudaMemcpyAsync(rhoD, drD, w * Ns, cudaMemcpyDeviceToHost, st))
    }
    CRF_TRY(cudaStreamSynchronize(st))
#undef CRF_TRY
    return CRF_OK;
}

}  // extern "C"
