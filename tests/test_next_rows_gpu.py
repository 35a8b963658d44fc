"""GPU parity of the SURVEY.md 8(f) rows built on the hot path: crf_rhs_pointwise (row 1: the fused right-hand-side
evaluation with its by-products rho, Wbar, c_pk), crf_production_rates_pair and crf_production_rates_jv (row 2: two
states per launch and the difference quotient of the Jacobian-vector product).  All through the C ABI, against the
oracle on the same seeded inputs, at BASELINE.json's tolerances (the quotient: the tolerance of two evaluations
divided by sigma)."""
import numpy as np
import pytest
import torch

from paper_2409_06404_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu

SMALL_N = {"C1": 512, "C2": 2 * 1024 + 333, "C3": 3 * 1024 + 77, "C4": 1024 + 301, "C5": 512 + 129}


@pytest.fixture(scope="module")
def binding():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2409_06404_b200 import binding as b
    b.lib()
    return b


def _np(d):
    return {k: (v.cpu().numpy() if v is not None else None) for k, v in d.items()}


def _check_rhs(out, ref, what):
    e = parity.assert_parity(out, ref, what)
    for key in ("cpk", "rho", "Wbar"):
        err = float(np.max(np.abs(out[key] - ref[key]) / np.abs(ref[key])))
        assert err <= parity.RTOL, f"{what}: {key} relative error {err:.3g}"
        e[key] = err / parity.RTOL
    return e


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5"])
@pytest.mark.parametrize("odd", [0, 1])
def test_rhs_pointwise(binding, oracle_mod, name, odd):
    desc = wl.make_mechanism(name)
    gm, om = binding.Mechanism(desc), oracle_mod.Oracle(desc)
    n = SMALL_N[name] + odd
    st = wl.make_state(name, n=n, total=n)
    d = parity.to_dev(st)
    out = _np(gm.rhs_pointwise(d["T"], d["p"], d["Y"]))
    e = _check_rhs(out, om.rhs_pointwise(**st), f"rhs {name} n={n}")
    print(name, n, {k: f"{v:.3g}" for k, v in e.items()})
    # the outputs shared with the three separate calls are the same numbers within the same tolerances, and the
    # by-products may be skipped
    out2 = _np(gm.rhs_pointwise(d["T"], d["p"], d["Y"], want_cpk=False))
    assert out2["cpk"] is None and np.array_equal(out2["omega"], out["omega"]) and np.array_equal(out2["cp"], out["cp"])


@pytest.mark.parametrize("opt", [dict(rates_kernel="staged"), dict(rates_kernel="generic"), dict(rates_kernel="group", rates_tmem=1),
                                 dict(rates_kernel="group", rates_PPL=1)],
                         ids=lambda o: ",".join(f"{k}={v}" for k, v in o.items()))
def test_rhs_pointwise_other_plans(binding, oracle_mod, opt):
    """Mechanisms without a warp-group plan take the separate kernels; u rows in shared memory and one point per lane
    emit the same by-products."""
    desc = wl.make_mechanism("C3")
    gm, om = binding.Mechanism(desc, options=opt), oracle_mod.Oracle(desc)
    n = 1025
    st = wl.make_state("C3", n=n, total=n)
    d = parity.to_dev(st)
    _check_rhs(_np(gm.rhs_pointwise(d["T"], d["p"], d["Y"])), om.rhs_pointwise(**st), f"rhs C3 {opt}")


def _two_states(name, n):
    a = wl.make_state(name, n=n, total=2 * n)
    b = wl.make_state(name, n=n, offset=n, total=2 * n)
    return a, b


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_pair_matches_oracle_and_single_calls(binding, oracle_mod, name):
    desc = wl.make_mechanism(name)
    gm = binding.Mechanism(desc, options=dict(rates_kernel="group"))
    om = oracle_mod.Oracle(desc)
    n = SMALL_N[name]
    a, b = _two_states(name, n)
    da, db = parity.to_dev(a), parity.to_dev(b)
    o1, q1, o2, q2 = gm.production_rates_pair(da["T"], da["p"], da["Y"], db["T"], db["p"], db["Y"])
    ref = om.production_rates_pair(a["T"], a["p"], a["Y"], b["T"], b["p"], b["Y"])
    for got, key, sk in ((o1, "omega", "S_omega"), (q1, "qdot", "S_q"), (o2, "omega2", "S_omega2"), (q2, "qdot2", "S_q2")):
        err = np.max(np.abs(got.cpu().numpy() - ref[key]) / (parity.RATE_TOL * ref[sk] + 1e-30))
        assert err <= 1.0, (name, key, err)
    # one launch for two states = two launches of the same kernel, bit for bit
    s1, sq1 = gm.production_rates(da["T"], da["p"], da["Y"])
    s2, sq2 = gm.production_rates(db["T"], db["p"], db["Y"])
    assert torch.equal(o1, s1) and torch.equal(q1, sq1) and torch.equal(o2, s2) and torch.equal(q2, sq2)


@pytest.mark.parametrize("name", ["C1", "C2"])
def test_pair_on_the_thread_kernel(binding, oracle_mod, name):
    """Small mechanisms (default plan: one thread per point, state in tensor memory): the thread evaluates the two states
    one after the other in one launch; bit-identical to two single calls, ragged n."""
    desc = wl.make_mechanism(name)
    gm, om = binding.Mechanism(desc), oracle_mod.Oracle(desc)
    info = gm.plan_info()
    assert info["rates_kernel"] == "thread" and info["rates_tmem_cols"] > 0, info
    n = 1000 + 37
    a, b = _two_states(name, n)
    da, db = parity.to_dev(a), parity.to_dev(b)
    o1, q1, o2, q2 = gm.production_rates_pair(da["T"], da["p"], da["Y"], db["T"], db["p"], db["Y"])
    s1, sq1 = gm.production_rates(da["T"], da["p"], da["Y"])
    s2, sq2 = gm.production_rates(db["T"], db["p"], db["Y"])
    assert torch.equal(o1, s1) and torch.equal(q1, sq1) and torch.equal(o2, s2) and torch.equal(q2, sq2)
    ref = om.production_rates_pair(a["T"], a["p"], a["Y"], b["T"], b["p"], b["Y"])
    assert np.max(np.abs(o2.cpu().numpy() - ref["omega2"]) / (parity.RATE_TOL * ref["S_omega2"] + 1e-30)) <= 1.0
    # the shared-memory version of the same kernel (rates_tmem = 1) meets the same tolerance
    g2 = binding.Mechanism(desc, options=dict(rates_tmem=1))
    assert g2.plan_info()["rates_tmem_cols"] == 0
    s3, _ = g2.production_rates(da["T"], da["p"], da["Y"])
    assert np.max(np.abs(s3.cpu().numpy() - ref["omega"]) / (parity.RATE_TOL * ref["S_omega"] + 1e-30)) <= 1.0


def test_pair_without_a_shared_launch(binding, oracle_mod):
    """A plan that cannot hold two states per lane answers the pair call with two launches: same numbers."""
    desc = wl.make_mechanism("C3")
    gm, om = binding.Mechanism(desc, options=dict(rates_kernel="staged")), oracle_mod.Oracle(desc)
    a, b = _two_states("C3", 777)
    da, db = parity.to_dev(a), parity.to_dev(b)
    o1, q1, o2, q2 = gm.production_rates_pair(da["T"], da["p"], da["Y"], db["T"], db["p"], db["Y"])
    ref = om.production_rates_pair(a["T"], a["p"], a["Y"], b["T"], b["p"], b["Y"])
    assert np.max(np.abs(o2.cpu().numpy() - ref["omega2"]) / (parity.RATE_TOL * ref["S_omega2"] + 1e-30)) <= 1.0
    assert np.max(np.abs(o1.cpu().numpy() - ref["omega"]) / (parity.RATE_TOL * ref["S_omega"] + 1e-30)) <= 1.0
    with pytest.raises(binding.CrfError, match="no warp-group plan"):
        gm.production_rates_jv(da["T"], da["p"], da["Y"], db["T"], db["p"], db["Y"], 1e-6)


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
@pytest.mark.parametrize("sigma", [1e-3, -1e-7])
def test_jv_difference_quotient(binding, oracle_mod, name, sigma):
    """(omega(y + sigma v) - omega(y)) / sigma, perturbation formed in the kernel: the direction is a seeded random
    vector scaled like the state (the perturbation factor of [17], would scale it the same way)."""
    desc = wl.make_mechanism(name)
    gm, om = binding.Mechanism(desc), oracle_mod.Oracle(desc)  # default plan: the call uses the warp-group plan
    n = SMALL_N[name] + 1
    st = wl.make_state(name, n=n, total=n)
    rng = np.random.default_rng(42)
    v = dict(dT=st["T"] * rng.uniform(-1, 1, n), dp=st["p"] * rng.uniform(-1, 1, n),
             dY=st["Y"] * rng.uniform(-1, 1, st["Y"].shape))
    d, dv = parity.to_dev(st), parity.to_dev(v)
    om_b, qd_b, Jo, Jq = gm.production_rates_jv(d["T"], d["p"], d["Y"], dv["dT"], dv["dp"], dv["dY"], sigma)
    ref = om.production_rates_jv(st["T"], st["p"], st["Y"], v["dT"], v["dp"], v["dY"], sigma)
    e = {}
    for got, key, sk in ((om_b, "omega", "S_omega"), (qd_b, "qdot", "S_q"), (Jo, "Jomega", "S_Jomega"), (Jq, "Jqdot", "S_Jqdot")):
        e[key] = float(np.max(np.abs(got.cpu().numpy() - ref[key]) / (parity.RATE_TOL * ref[sk] + 1e-30 / abs(sigma))))
        assert e[key] <= 1.0, (name, key, e)
    print(name, sigma, {k: f"{x:.3g}" for k, x in e.items()})
    # the quotient alone (no base outputs), and without a pressure perturbation
    _, _, Jo2, Jq2 = gm.production_rates_jv(d["T"], d["p"], d["Y"], dv["dT"], dv["dp"], dv["dY"], sigma, base=False)
    assert torch.equal(Jo2, Jo) and torch.equal(Jq2, Jq)
    _, _, Jo3, _ = gm.production_rates_jv(d["T"], d["p"], d["Y"], dv["dT"], None, dv["dY"], sigma)
    ref3 = om.production_rates_jv(st["T"], st["p"], st["Y"], v["dT"], np.zeros(n), v["dY"], sigma)
    assert np.max(np.abs(Jo3.cpu().numpy() - ref3["Jomega"]) / (parity.RATE_TOL * ref3["S_Jomega"] + 1e-30 / abs(sigma))) <= 1.0


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5"])
def test_jv_against_a_given_base(binding, oracle_mod, name):
    """crf_production_rates_jv_base: omega(y), qdot(y) are inputs (what an integrator has in hand), only
    the perturbed state is evaluated: bit for bit the quotient of crf_production_rates_jv for the same base values, within
    tolerance of the oracle's quotient, also under a plan with one point per lane (which the two-state call declines)."""
    desc = wl.make_mechanism(name)
    gm, om = binding.Mechanism(desc), oracle_mod.Oracle(desc)
    n = SMALL_N[name] + 1  # odd: the ragged tail of the two-points-per-lane rows
    st = wl.make_state(name, n=n, total=n)
    rng = np.random.default_rng(43)
    v = dict(dT=st["T"] * rng.uniform(-1, 1, n), dp=st["p"] * rng.uniform(-1, 1, n),
             dY=st["Y"] * rng.uniform(-1, 1, st["Y"].shape))
    d, dv = parity.to_dev(st), parity.to_dev(v)
    sigma = 1e-6
    om_b, qd_b, Jo, Jq = gm.production_rates_jv(d["T"], d["p"], d["Y"], dv["dT"], dv["dp"], dv["dY"], sigma)
    om_s, qd_s = gm.production_rates(d["T"], d["p"], d["Y"])
    assert torch.equal(om_s, om_b) and torch.equal(qd_s, qd_b)
    keep = (om_s.clone(), qd_s.clone())
    Jo4, Jq4 = gm.production_rates_jv_base(d["T"], d["p"], d["Y"], dv["dT"], dv["dp"], dv["dY"], sigma, om_s, qd_s)
    assert torch.equal(Jo4, Jo) and torch.equal(Jq4, Jq)
    assert torch.equal(om_s, keep[0]) and torch.equal(qd_s, keep[1])  # the base values are inputs: untouched
    ref = om.production_rates_jv(st["T"], st["p"], st["Y"], v["dT"], v["dp"], v["dY"], sigma)
    for got, key, sk in ((Jo4, "Jomega", "S_Jomega"), (Jq4, "Jqdot", "S_Jqdot")):
        assert np.max(np.abs(got.cpu().numpy() - ref[key]) / (parity.RATE_TOL * ref[sk] + 1e-30 / abs(sigma))) <= 1.0, (name, key)
    # no pressure perturbation
    Jo5, _ = gm.production_rates_jv_base(d["T"], d["p"], d["Y"], dv["dT"], None, dv["dY"], sigma, om_s, qd_s)
    ref5 = om.production_rates_jv(st["T"], st["p"], st["Y"], v["dT"], np.zeros(n), v["dY"], sigma)
    assert np.max(np.abs(Jo5.cpu().numpy() - ref5["Jomega"]) / (parity.RATE_TOL * ref5["S_Jomega"] + 1e-30 / abs(sigma))) <= 1.0
    # one point per lane in the warp-group kernel
    g1 = binding.Mechanism(desc, options=dict(rates_kernel="group", rates_PPL=1))
    b1 = g1.production_rates(d["T"], d["p"], d["Y"])
    Jo6, Jq6 = g1.production_rates_jv_base(d["T"], d["p"], d["Y"], dv["dT"], dv["dp"], dv["dY"], sigma, *b1)
    for got, key, sk in ((Jo6, "Jomega", "S_Jomega"), (Jq6, "Jqdot", "S_Jqdot")):
        assert np.max(np.abs(got.cpu().numpy() - ref[key]) / (parity.RATE_TOL * ref[sk] + 1e-30 / abs(sigma))) <= 1.0, (name, key, "PPL=1")
    # a fall-back kernel declines
    g2 = binding.Mechanism(desc, options=dict(rates_kernel="staged"))
    with pytest.raises(binding.CrfError, match="fall-back"):
        g2.production_rates_jv_base(d["T"], d["p"], d["Y"], dv["dT"], dv["dp"], dv["dY"], sigma, *b1)


def test_new_calls_reject_bad_arguments(binding):
    desc = wl.make_mechanism("C1")
    gm = binding.Mechanism(desc)
    st = parity.to_dev(wl.make_state("C1", n=64, total=64))
    with pytest.raises(binding.CrfError, match="sigma"):
        gm.production_rates_jv(st["T"], st["p"], st["Y"], st["T"], st["p"], st["Y"], 0.0)
    L = binding.lib()
    z = torch.zeros(64 * 9 + 8, dtype=torch.float64, device="cuda")
    args = [gm._h, st["T"].data_ptr(), st["p"].data_ptr(), st["Y"].data_ptr(), 64]
    outs = [z.data_ptr()] * 10
    assert L.crf_rhs_pointwise(*args, *outs) == 0
    outs[0] = z.data_ptr() + 8
    assert L.crf_rhs_pointwise(*args, *outs) == -1  # misaligned
    outs[0] = None
    assert L.crf_rhs_pointwise(*args, *outs) == -1  # omega is required
    assert L.crf_rhs_pointwise(gm._h, st["T"].data_ptr(), st["p"].data_ptr(), st["Y"].data_ptr(), 0, *([None] * 10)) == 0


@pytest.mark.parametrize("name", ["C2", "C5"])
def test_next_rows_at_full_size_sampled(binding, oracle_mod, name):
    """BASELINE.json's full sizes, in the launch configurations `bench.py --path rhs | jv | sem` times: sampled points
    (the first and last, block boundaries, random ones) and sampled elements against the oracle, plus properties of the
    whole fields."""
    from oracle import sem_oracle
    desc = wl.make_mechanism(name)
    gm, om = binding.Mechanism(desc), oracle_mod.Oracle(desc)
    n = wl.config_points(name)
    st = wl.make_state(name)
    d = parity.to_dev(st)
    rng = np.random.default_rng(321)
    idx = np.unique(np.concatenate(([0, 1, 63, 64, 127, 128, n - 2, n - 1], rng.integers(0, n, 248))))
    sub = dict(T=st["T"][idx], p=st["p"][idx], Y=np.ascontiguousarray(st["Y"][:, idx]))

    def take(t):
        return None if t is None else (t[:, idx] if t.dim() == 2 else t[idx]).cpu().numpy()

    # crf_rhs_pointwise
    rhs = gm.rhs_pointwise(d["T"], d["p"], d["Y"])
    _check_rhs({k: take(v) for k, v in rhs.items()}, om.rhs_pointwise(**sub), f"rhs {name} full")
    assert bool(torch.isfinite(rhs["rho"]).all()) and bool((rhs["rho"] > 0).all()) and bool((rhs["Wbar"] > 0).all())

    # crf_production_rates_jv
    v = {k: d[k] * (2 * torch.rand(d[k].shape, dtype=torch.float64, device="cuda", generator=torch.Generator("cuda").manual_seed(5)) - 1)
         for k in ("T", "p", "Y")}
    sigma = 1e-6
    _, _, Jo, Jq = gm.production_rates_jv(d["T"], d["p"], d["Y"], v["T"], v["p"], v["Y"], sigma)
    vs = {k: take(t) for k, t in v.items()}
    ref = om.production_rates_jv(sub["T"], sub["p"], sub["Y"], vs["T"], vs["p"], vs["Y"], sigma)
    assert np.max(np.abs(take(Jo) - ref["Jomega"]) / (parity.RATE_TOL * ref["S_Jomega"] + 1e-30 / sigma)) <= 1.0
    assert np.max(np.abs(take(Jq) - ref["Jqdot"]) / (parity.RATE_TOL * ref["S_Jqdot"] + 1e-30 / sigma)) <= 1.0
    assert bool(torch.isfinite(Jo).all())
    # crf_production_rates_jv_base on the whole field: the same quotient, bit for bit, from the base values of the plain call
    Jo2, Jq2 = gm.production_rates_jv_base(d["T"], d["p"], d["Y"], v["T"], v["p"], v["Y"], sigma, rhs["omega"], rhs["qdot"])
    assert torch.equal(Jo2, Jo) and torch.equal(Jq2, Jq)
    del Jo, Jo2, v

    # crf_sem_diffusion on every element, sampled elements against the oracle (the operator is element-local)
    nel = n // 512
    h3 = np.random.default_rng(7).uniform(0.2e-3, 1.5e-3, (nel, 3))
    dY, dT = gm.sem_diffusion(torch.from_numpy(h3).cuda(), d["T"], rhs["Wbar"], d["Y"], rhs["lam"], rhs["rhoD"])
    els = np.unique(np.concatenate(([0, 1, nel - 1], rng.integers(0, nel, 5))))
    pts = (els[:, None] * 512 + np.arange(512)[None, :]).reshape(-1)
    pt = torch.from_numpy(pts).cuda()
    args = (desc["W"], h3[els], st["T"][pts], rhs["Wbar"][pt].cpu().numpy(), np.ascontiguousarray(st["Y"][:, pts]),
            rhs["lam"][pt].cpu().numpy(), rhs["rhoD"][:, pt].cpu().numpy())
    sr, ss = sem_oracle.sem_diffusion(*args), sem_oracle.sem_diffusion_scale(*args)
    assert np.max(np.abs(dY[:, pt].cpu().numpy() - sr["dY"]) / (1e-12 * ss["dY"] + 1e-300)) <= 1.0
    assert np.max(np.abs(dT[pt].cpu().numpy() - sr["dT"]) / (1e-12 * ss["dT"] + 1e-300)) <= 1.0
    assert bool(torch.isfinite(dY).all()) and bool(torch.isfinite(dT).all())
