"""GPU parity tests proper: the CUDA path, called through the C ABI (ctypes binding), against
the CPU oracle on the same seeded inputs.  Tolerances are BASELINE.json's (tests/parity.py).

* element by element at sizes the oracle finishes in seconds, spanning several thread blocks
  and a ragged (odd) tail, for the five mechanisms C1..C5 in both h_f modes of the generator;
* at BASELINE.json's full sizes, in the launch configuration bench.py times, on sampled
  points (the path is pointwise, so the oracle evaluates the sampled columns one by one);
* edge cases: n = 0, n = 1, odd n, pure species (the D_kk guard), T exactly at T_mid,
  misaligned and null pointers, a non-default stream.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2409_06404_b200 import workloads as wl
from tests import parity
from tests.helpers import P_REF, rxn, tiny_mech

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2409_06404_b200 import binding as b
    b.lib()  # raises if libcrf.so is missing: there is no fallback
    return b


_cache = {}


def _mech_pair(binding, oracle_mod, name, hf="uniform"):
    key = (name, hf)
    if key not in _cache:
        desc = wl.make_mechanism(name, hf=hf)
        _cache[key] = (desc, binding.Mechanism(desc), oracle_mod.Oracle(desc))
    return _cache[key]


SMALL_N = {"C1": 512, "C2": 2 * 1024 + 333, "C3": 3 * 1024 + 77, "C4": 1024 + 301, "C5": 512 + 129}


@pytest.mark.parametrize("hf", ["uniform", "group"])
@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5"])
def test_elementwise_small(binding, oracle_mod, name, hf):
    desc, gm, om = _mech_pair(binding, oracle_mod, name, hf)
    n = SMALL_N[name]
    st = wl.make_state(name, n=n, total=n)
    e = parity.assert_parity(parity.run_gpu(gm, st), parity.run_oracle(om, st), f"{name}/{hf} n={n}")
    print(name, hf, {k: f"{v:.3g}" for k, v in e.items()})


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_full_size_sampled(binding, oracle_mod, name):
    """Full BASELINE.json size, device-resident, same calls bench.py times; 384 sampled points
    (always including the first and last point and a block boundary) checked against the oracle."""
    desc, gm, om = _mech_pair(binding, oracle_mod, name)
    n = wl.config_points(name)
    st = wl.make_state(name)
    gpu = parity.run_gpu(gm, st)
    rng = np.random.default_rng(123)
    idx = np.unique(np.concatenate(([0, 1, 127, 128, 255, 256, n - 2, n - 1], rng.integers(0, n, 376))))
    sub = dict(T=st["T"][idx], p=st["p"][idx], Y=np.ascontiguousarray(st["Y"][:, idx]))
    gsub = {k: (v[:, idx] if v.ndim == 2 else v[idx]) for k, v in gpu.items()}
    parity.assert_parity(gsub, parity.run_oracle(om, sub), f"{name} full n={n}")
    # properties that hold at any size, over the whole field
    for key in ("cp", "mu", "lam", "rhoD"):
        assert np.all(np.isfinite(gpu[key])) and np.all(gpu[key] > 0.0), key
    assert np.all(np.isfinite(gpu["omega"])) and np.all(np.isfinite(gpu["qdot"])) and np.all(np.isfinite(gpu["h"]))
    # mass conservation sum_k W_k omega_k = 0 within the rate tolerance scale of the sampled points
    W = np.asarray(desc["W"])
    ref = om.production_rates(**sub)
    assert np.all(np.abs(W @ gsub["omega"]) <= 1e-10 * (W @ ref["S_omega"]) + 1e-30)


@pytest.mark.parametrize("n", [0, 1, 2, 3, 31, 33, 127, 129, 255, 257])
def test_ragged_sizes(binding, oracle_mod, n):
    desc, gm, om = _mech_pair(binding, oracle_mod, "C3")
    st = wl.make_state("C3", n=n, total=max(n, 1))
    if n == 0:
        d = parity.to_dev(st)
        gm.thermo(d["T"], d["p"], d["Y"])
        gm.production_rates(d["T"], d["p"], d["Y"])
        gm.mix_transport(d["T"], d["p"], d["Y"])
        torch.cuda.synchronize()
        return
    parity.assert_parity(parity.run_gpu(gm, st), parity.run_oracle(om, st), f"C3 n={n}")


def test_outputs_do_not_spill_past_n(binding, oracle_mod):
    """Rows of the species-major outputs are written for exactly n points (guard cells untouched)."""
    desc, gm, om = _mech_pair(binding, oracle_mod, "C1")
    n, pad = 130, 6
    st = wl.make_state("C1", n=n)
    d = parity.to_dev(st)
    Ns = gm.Ns
    big = torch.full((Ns * n + pad,), -777.0, dtype=torch.float64, device="cuda")
    big2 = torch.full((Ns * n + pad,), -777.0, dtype=torch.float64, device="cuda")
    qd = torch.full((n + pad,), -777.0, dtype=torch.float64, device="cuda")
    gm.production_rates(d["T"], d["p"], d["Y"], omega=big[: Ns * n].view(Ns, n), qdot=qd[:n])
    gm.mix_transport(d["T"], d["p"], d["Y"], rhoD=big2[: Ns * n].view(Ns, n))
    torch.cuda.synchronize()
    assert torch.all(big[Ns * n:] == -777.0) and torch.all(big2[Ns * n:] == -777.0) and torch.all(qd[n:] == -777.0)
    assert not torch.any(big[: Ns * n] == -777.0)


def test_pure_species_and_tmid(binding, oracle_mod):
    """Degenerate cases: each species pure (sum_{j!=k} X_j/D_jk == 0 -> rho D_kk), Y with exact
    zeros, and T exactly at (and one ulp around) each species' T_mid."""
    desc, gm, om = _mech_pair(binding, oracle_mod, "C3")
    Ns = gm.Ns
    tm = np.asarray(desc["nasa_Tmid"])
    Tm = np.concatenate((tm, np.nextafter(tm, 0.0), np.nextafter(tm, 1e9)))
    n = Ns + Tm.size
    Y = np.zeros((Ns, n))
    Y[np.arange(Ns), np.arange(Ns)] = 1.0
    rng = np.random.default_rng(3)
    Yr = rng.dirichlet(np.full(Ns, 0.5), size=Tm.size).T
    Yr[rng.random(Yr.shape) < 0.3] = 0.0
    Yr[0] += 1e-3
    Y[:, Ns:] = Yr / Yr.sum(axis=0)
    T = np.concatenate((rng.uniform(300, 2500, Ns), Tm))
    st = dict(T=T, p=np.full(n, 2.5e5), Y=np.ascontiguousarray(Y))
    gpu, ref = parity.run_gpu(gm, st), parity.run_oracle(om, st)
    parity.assert_parity(gpu, ref, "pure species / T_mid")
    # the guard really was hit: pure-species rows equal rho D_kk in the oracle
    assert np.all(ref["rhoD"][np.arange(Ns), np.arange(Ns)] > 0)


def test_hand_built_mechanism(binding, oracle_mod):
    """A three-slot reaction (2A + B <=> C + D + E is outside the generator's forms), a reaction with
    coefficient 2 and a falloff reaction without listed efficiencies."""
    W = [2.0, 32.0, 18.0, 17.0, 1.0, 28.0]
    troe = dict(A0=1e17, beta0=-0.5, Ea0=5.0, alpha=0.6, T3=100.0, T1=2000.0, T2=5000.0)
    rx = [rxn([(0, 2), (1, 1)], [(2, 1), (3, 1), (4, 1)], A=1e11, beta=0.3, Ea=20.0),
          rxn([(3, 2)], [(2, 1), (4, 2)], A=1e9, beta=1.0, Ea=40.0),
          rxn([(3, 1), (4, 1)], [(2, 1)], A=1e13, beta=-0.2, Ea=3.0, type="falloff", eff={}, troe=troe),
          rxn([(4, 2)], [(0, 1)], A=1e16, beta=-1.0, Ea=0.0, type="three_body", eff={0: 2.5, 2: 12.0})]
    desc = tiny_mech(W, rx)
    gm, om = binding.Mechanism(desc), oracle_mod.Oracle(desc)
    rng = np.random.default_rng(0)
    n = 257
    Y = rng.dirichlet(np.ones(6), size=n).T
    st = dict(T=rng.uniform(300, 2500, n), p=rng.uniform(1e4, 1e7, n), Y=np.ascontiguousarray(Y))
    parity.assert_parity(parity.run_gpu(gm, st), parity.run_oracle(om, st), "hand-built")


def test_species_thermo(binding, oracle_mod):
    desc, gm, om = _mech_pair(binding, oracle_mod, "C4")
    T = np.random.default_rng(1).uniform(250, 3200, 1001)
    cpk, hk, sk = (t.cpu().numpy() for t in gm.thermo_species(torch.from_numpy(T).cuda()))
    ref = om.thermo_species(T)
    np.testing.assert_allclose(cpk, ref["cpk"], rtol=1e-12)
    np.testing.assert_allclose(sk, ref["sk"], rtol=1e-12)
    assert np.all(np.abs(hk - ref["hk"]) <= 1e-12 * np.maximum(np.abs(ref["hk"]), 1e-3 * ref["cpk"] * T))


def test_stream_and_errors(binding, oracle_mod):
    desc, gm, om = _mech_pair(binding, oracle_mod, "C1")
    st = wl.make_state("C1", n=512)
    ref = parity.run_oracle(om, st)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        gpu = parity.run_gpu(gm, st)
    parity.assert_parity(gpu, ref, "side stream")
    d = parity.to_dev(st)
    L = binding.lib()
    n = 512
    out = torch.empty(9 * n + 2, dtype=torch.float64, device="cuda")
    q = torch.empty(n, dtype=torch.float64, device="cuda")
    args = (gm._h, d["T"].data_ptr(), d["p"].data_ptr(), d["Y"].data_ptr())
    assert L.crf_production_rates(*args, n, out.data_ptr() + 8, q.data_ptr()) == -1  # misaligned
    assert b"aligned" in L.crf_last_error()
    assert L.crf_production_rates(*args, n, None, q.data_ptr()) == -1                # null
    assert L.crf_production_rates(*args, -5, out.data_ptr(), q.data_ptr()) == -1     # negative n
    assert L.crf_mix_transport(None, d["T"].data_ptr(), d["p"].data_ptr(), d["Y"].data_ptr(), n,
                               q.data_ptr(), q.data_ptr(), out.data_ptr()) == -1
    with pytest.raises(binding.CrfError):
        gm.thermo(d["T"].float(), d["p"], d["Y"])


def test_step_host_matches_device_calls(binding, oracle_mod):
    """crf_step_host (host buffers, chunked pipeline) gives bit-identical results to the device calls
    on a size that spans several chunks with a ragged last chunk."""
    desc, gm, om = _mech_pair(binding, oracle_mod, "C3")
    n = 2 * 524288 + 12345  # (a chunk of this mechanism is 524288 points)
    st = wl.make_state("C3", n=n)
    gpu = parity.run_gpu(gm, st)
    host = {k: torch.from_numpy(v).pin_memory() for k, v in st.items()}
    out = gm.step_host(host["T"], host["p"], host["Y"])
    for key in ("cp", "h", "omega", "qdot", "mu", "lam", "rhoD"):
        np.testing.assert_array_equal(out[key].numpy(), gpu[key], err_msg=key)
    idx = np.random.default_rng(5).integers(0, n, 256)
    sub = dict(T=st["T"][idx], p=st["p"][idx], Y=np.ascontiguousarray(st["Y"][:, idx]))
    hsub = {k: (v.numpy()[:, idx] if v.ndim == 2 else v.numpy()[idx]) for k, v in out.items()}
    parity.assert_parity(hsub, parity.run_oracle(om, sub), "step_host")


def test_step_host_output_groups(binding, oracle_mod):
    """crf_step_host computes and copies only the groups of outputs that are asked for."""
    desc, gm, om = _mech_pair(binding, oracle_mod, "C3")
    n = 600000  # more than one pipeline chunk
    st = wl.make_state("C3", n=n, total=n)
    host = {k: torch.from_numpy(v) for k, v in st.items()}
    full = gm.step_host(host["T"], host["p"], host["Y"])
    part = dict(omega=torch.empty(gm.Ns, n, dtype=torch.float64), qdot=torch.empty(n, dtype=torch.float64))
    gm.step_host(host["T"], host["p"], host["Y"], part)
    assert torch.equal(part["omega"], full["omega"]) and torch.equal(part["qdot"], full["qdot"])
    with pytest.raises(binding.CrfError, match="together"):
        gm.step_host(host["T"], host["p"], host["Y"], dict(omega=part["omega"]))
    with pytest.raises(binding.CrfError, match="no output"):
        gm.step_host(host["T"], host["p"], host["Y"], {})


def test_step_host_f32_outputs(binding, oracle_mod):
    """crf_step_host_f32: double arithmetic, outputs rounded once to float on the device: every value is the float
    nearest to the double-precision result of crf_step_host (bit for bit), hence within 2^-24 of the oracle."""
    desc, gm, om = _mech_pair(binding, oracle_mod, "C3")
    n = 540000 + 3  # (two chunks, the second ragged)
    st = wl.make_state("C3", n=n, total=n)
    host = {k: torch.from_numpy(v) for k, v in st.items()}
    full = gm.step_host(host["T"], host["p"], host["Y"])
    out32 = {k: torch.empty(v.shape, dtype=torch.float32) for k, v in full.items()}
    gm.step_host(host["T"], host["p"], host["Y"], out32)
    for k, v in full.items():
        assert torch.equal(out32[k], v.to(torch.float32)), k
    ref = om.mix_transport(**{k: v[..., :512] for k, v in st.items()})
    assert np.max(np.abs(out32["rhoD"][:, :512].numpy() - ref["rhoD"]) / ref["rhoD"]) <= 2.0 ** -24 * 1.001
    part = dict(omega=torch.empty(gm.Ns, n, dtype=torch.float32), qdot=torch.empty(n, dtype=torch.float32))
    gm.step_host(host["T"], host["p"], host["Y"], part)
    assert torch.equal(part["omega"], out32["omega"])


def test_fp64_probe(binding):
    r = binding.fp64_probe(2048)
    assert 1e12 < r < 4e13, r  # B200: 148 SM x 64 lanes x ~1.9 GHz = 1.8e13 FP64 instr/s nominal


PLAN_OVERRIDES = [
    dict(transport_kernel="tiled", transport_PPL=2),       # two points per lane in the tiled transport kernel
    dict(transport_kernel="tiled", transport_W=4),         # rounds split over fewer warps than tiles
    dict(transport_kernel="tiled", transport_W=1, transport_PPL=2),
    dict(transport_kernel="tiled", transport_panel=1),     # one column block per Wilke panel (most stage steps)
    dict(transport_kernel="tiled", transport_TS=8),        # species blocks of 8 in both phases
    dict(transport_kernel="tiled", transport_TS=7),        # blocks of 7 (the automatic choice for C3 and C4; C5: 17 blocks, split rounds)
    dict(transport_kernel="tiled", transport_TS=7, transport_PPL=2),
    dict(transport_kernel="tiled", transport_TS=7, transport_W=2, transport_panel=2),  # Wilke panels that end off a multiple of 4
    dict(rates_kernel="group", rates_W=8, rates_PPL=1),
    dict(rates_kernel="group", rates_W=4, rates_PPL=2, rates_Rc=32),   # many small chunks
    dict(rates_kernel="group", rates_W=16, rates_PPL=2),
    dict(rates_kernel="group", rates_tmem=1),              # u rows in shared memory (the path of Ns > 127)
    dict(rates_kernel="group", rates_tmem=2),              # u rows in tensor memory, required
    dict(rates_kernel="group", rates_W=16, rates_PPL=1, rates_tmem=2),
    dict(rates_kernel="staged"),                           # log-space K_c kernel (the automatic fall-back)
    dict(rates_kernel="generic"),                          # one thread per point, libm
    dict(rates_kernel="thread"),                           # one thread per point, product form (default for Ns <= 12)
    dict(transport_kernel="generic"),
    dict(thermo_sets=1),                                   # crf_thermo: every lane reads the NASA-7 set of its own range
    dict(thermo_sets=2),                                   # both sets at uniform addresses (the default)
    dict(transport_kernel="small"),
]


def _admits(name, opt):
    Ns = wl.CONFIGS[name]["Ns"]
    if opt.get("rates_kernel") == "thread" and Ns > 24:
        return False
    if opt.get("rates_kernel") == "group" and opt.get("rates_W") and (Ns + opt["rates_W"] - 1) // opt["rates_W"] > 16:
        return False
    if opt.get("rates_kernel") == "group" and Ns <= 12 and not opt.get("rates_W"):
        pass  # (the warp-group kernel also takes small mechanisms on request)
    if opt.get("transport_kernel") == "small" and Ns > 16:
        return False
    if opt.get("transport_kernel") == "tiled" and Ns < 17:
        return False
    return True


@pytest.mark.parametrize("opt", PLAN_OVERRIDES, ids=lambda o: ",".join(f"{k}={v}" for k, v in o.items()))
@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_plan_overrides(binding, oracle_mod, name, opt):
    """The kernel plans are chosen in crf_mech_create; crf_mech_create_ex (crf_diag.h) selects the other kernels and
    template instances (warps per point group, points per lane, chunk size, fall-back kernels): each must meet the
    same tolerances on a ragged size, and a request the mechanism does not admit must fail, not fall back."""
    desc = wl.make_mechanism(name)
    if not _admits(name, opt):
        with pytest.raises(binding.CrfError):
            binding.Mechanism(desc, options=opt)
        return
    try:
        gm = binding.Mechanism(desc, options=opt)
    except binding.CrfError as err:
        # an explicit warps-per-group request may not fit the shared-memory budget of this mechanism: refused, never
        # silently replaced (which kernel ran is asserted below for every request that is honoured)
        assert "does not admit" in str(err) and opt.get("rates_W"), (opt, err)
        return
    om = oracle_mod.Oracle(desc)
    info = gm.plan_info()
    for k, v in opt.items():
        if k not in ("rates_Rc", "transport_panel", "rates_tmem"):
            assert info[k] == v, (k, info)
    if "rates_tmem" in opt:
        assert (info["rates_tmem_cols"] > 0) == (opt["rates_tmem"] == 2), info
    n = SMALL_N[name] + 2
    st = wl.make_state(name, n=n, total=n)
    parity.assert_parity(parity.run_gpu(gm, st), parity.run_oracle(om, st), f"{name} {opt} n={n}")


BIG = {"Ns160": dict(seed=5, elements=("C", "H", "O", "N"), Ns=160, Nr=900, N3=60, Nt=40, ndup=0, cmax=3, eff_all=False),
       "Ns220": dict(seed=6, elements=("C", "H", "O", "N"), Ns=220, Nr=1200, N3=80, Nt=60, ndup=6, cmax=3, eff_all=False)}


@pytest.mark.parametrize("which", ["Ns160", "Ns220"])
def test_mechanisms_larger_than_C5(binding, oracle_mod, which):
    """crf_mech_create accepts up to CRF_MAX_SPECIES = 220 species: above C5 (118) the rates plan runs under a
    tighter shared-memory budget (one point per lane, more chunks) and the tiled transport kernel has up to 28
    species blocks.  Same tolerances, ragged size; the automatic plan must be a fast kernel, not the generic one."""
    desc = wl.make_mechanism(None, **BIG[which])
    gm, om = binding.Mechanism(desc), oracle_mod.Oracle(desc)
    info = gm.plan_info()
    assert info["rates_kernel"] == "group" and info["transport_kernel"] == "tiled", info
    n = 3 * 64 + 37
    st = wl.make_state("C5", n=n, Ns=BIG[which]["Ns"])
    parity.assert_parity(parity.run_gpu(gm, st), parity.run_oracle(om, st), f"{which} n={n} {info}")
    with pytest.raises(binding.CrfError):  # one species more than the limit
        binding.Mechanism(wl.make_mechanism(None, **dict(BIG["Ns220"], Ns=221)))


def _far_from_equilibrium_mechanism():
    """Formation enthalpies so far apart that the product form of 1/K_c (numerator and denominator formed
    separately) would leave the double range at the cold end of the validated window: the two reactants sit
    1.2e5 K (1000 kJ/mol) above the products, so at 250 K the numerator alone is 2^1385."""
    from tests.helpers import const_cp_nasa
    W = [10.0, 12.0, 9.0, 13.0, 28.0]
    nasa = np.array([const_cp_nasa(3.5, 1.2e5, 4.0), const_cp_nasa(4.0, 1.2e5, 5.0), const_cp_nasa(3.8, 0.0, 6.0),
                     const_cp_nasa(4.2, -2.0e3, 3.0), const_cp_nasa(3.5, 0.0, 5.0)])
    rx = [rxn([(0, 1), (1, 1)], [(2, 1), (3, 1)], A=1e12, beta=0.5, Ea=10.0),
          rxn([(0, 2)], [(2, 1), (3, 1)], A=1e10, beta=0.0, Ea=30.0, type="three_body", eff={4: 2.0}),
          rxn([(2, 1), (3, 1)], [(1, 2)], A=1e9, beta=1.0, Ea=5.0)]   # the same gap uphill: K_c underflows towards 0
    return tiny_mech(W, rx, nasa=(nasa, nasa))


def test_automatic_fallback_to_log_space_kernel(binding, oracle_mod):
    """No option is passed: crf_mech_create itself must notice that the product form of K_c is out of range and pick
    the log-space kernel (rates_staged.cu); requesting the product-form kernels for this mechanism must fail."""
    desc = _far_from_equilibrium_mechanism()
    gm, om = binding.Mechanism(desc), oracle_mod.Oracle(desc)
    assert gm.plan_info()["rates_kernel"] == "staged", gm.plan_info()
    for kernel in ("group", "thread"):
        with pytest.raises(binding.CrfError):
            binding.Mechanism(desc, options=dict(rates_kernel=kernel))
    rng = np.random.default_rng(8)
    n = 333
    # (reaction 3 runs uphill by the same gap: its K_c is 1e-100 at 1000 K, so k_r = k_f/K_c is huge but finite
    # above ~700 K; below that the oracle's own K_c underflows to 0 and the definition gives inf - not a test case)
    st = dict(T=rng.uniform(800.0, 2500.0, n), p=rng.uniform(5e4, 5e6, n),
              Y=np.ascontiguousarray(rng.dirichlet(np.ones(5), size=n).T))
    ref = parity.run_oracle(om, st)
    assert np.all(np.isfinite(ref["omega"]))
    parity.assert_parity(parity.run_gpu(gm, st), ref, "far from equilibrium (automatic staged kernel)")
    gg = binding.Mechanism(desc, options=dict(rates_kernel="generic"))
    parity.assert_parity(parity.run_gpu(gg, st), ref, "far from equilibrium (generic kernel)")


def test_mechanism_without_reactions(binding, oracle_mod):
    """Nr = 0 (a transport/thermo-only mechanism): no rates plan exists, crf_production_rates runs the generic kernel
    and returns exact zeros."""
    desc = tiny_mech([2.0, 32.0, 18.0, 28.0], [])
    gm, om = binding.Mechanism(desc), oracle_mod.Oracle(desc)
    assert gm.plan_info()["rates_kernel"] == "generic"
    rng = np.random.default_rng(2)
    n = 97
    st = dict(T=rng.uniform(300, 2500, n), p=np.full(n, P_REF), Y=np.ascontiguousarray(rng.dirichlet(np.ones(4), size=n).T))
    gpu = parity.run_gpu(gm, st)
    assert np.all(gpu["omega"] == 0.0) and np.all(gpu["qdot"] == 0.0)
    parity.assert_parity(gpu, parity.run_oracle(om, st), "Nr = 0")


TROE_SETS = {
    "chemkin_3_parameter": dict(alpha=0.5, T3=1e-30, T1=1e30, T2=1e30),      # 'TROE/0.5 1E-30 1E30/' + missing T2
    "T2_infinite": dict(alpha=0.7, T3=150.0, T1=1800.0, T2=float("inf")),
    "T2_huge": dict(alpha=0.62, T3=1e-30, T1=900.0, T2=1e300),
    "lindemann_inside_troe": dict(alpha=1.0, T3=1e300, T1=1e300, T2=1e300),  # F_cent = 1 -> F = 1
    "T3_infinite": dict(alpha=0.4, T3=float("inf"), T1=700.0, T2=4000.0),
}


@pytest.mark.parametrize("kernel", ["auto", "group", "staged", "generic", "thread"])
@pytest.mark.parametrize("which", sorted(TROE_SETS))
def test_troe_switched_off_terms(binding, oracle_mod, which, kernel):
    """Chemkin mechanisms switch Troe terms off with T3 = 1e-30, T1 = 1e30 and a missing (or 1e30 / infinite) T2:
    the arguments of the three exponentials of F_cent then reach -1e33 or -inf.  Every rates kernel must return what
    the definition gives (the terms are 0, alpha and 0) instead of reading garbage exponent bits."""
    W = [2.0, 32.0, 34.0, 17.0, 28.0]
    troe = dict(A0=3e17, beta0=-0.8, Ea0=2.0, **TROE_SETS[which])
    rx = [rxn([(3, 2)], [(2, 1)], A=2e13, beta=-0.3, Ea=1.0, type="falloff", eff={0: 2.0, 4: 0.7}, troe=troe),
          rxn([(0, 1), (1, 1)], [(3, 2)], A=1e11, beta=0.5, Ea=60.0),
          rxn([(3, 1), (0, 1)], [(2, 1)], A=5e12, beta=0.0, Ea=8.0, type="falloff", eff={}, troe=dict(troe, A0=1e16))]
    desc = tiny_mech(W, rx)
    gm, om = binding.Mechanism(desc, options=dict(rates_kernel=kernel)), oracle_mod.Oracle(desc)
    rng = np.random.default_rng(4)
    n = 161
    st = dict(T=rng.uniform(280, 3000, n), p=10.0 ** rng.uniform(3.5, 7.0, n),
              Y=np.ascontiguousarray(rng.dirichlet(np.ones(5), size=n).T))
    ref = parity.run_oracle(om, st)
    assert np.all(np.isfinite(ref["omega"])) and np.any(ref["omega"] != 0.0)
    parity.assert_parity(parity.run_gpu(gm, st), ref, f"Troe {which} / {kernel}")


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_extreme_states(binding, oracle_mod, name):
    """The corners of the range the kernels are specified for (crf_mech_create admits the product form of
    K_c for 250 K <= T <= 5000 K): very cold and very hot points, low and high pressure, mass fractions
    with exact zeros, a dominant species and traces down to 1e-30, next to ordinary points in the same warp."""
    desc, gm, om = _mech_pair(binding, oracle_mod, name)
    Ns = gm.Ns
    rng = np.random.default_rng(11)
    Ts = np.array([255.0, 300.0, 650.0, 1000.0, 1800.0, 3000.0, 4200.0, 4950.0])
    ps = np.array([1.0e3, 1.0e5, 1.0e7])
    T, p = (a.ravel() for a in np.meshgrid(Ts, ps, indexing="ij"))
    T, p = np.tile(T, 5), np.tile(p, 5)  # 120 points: several warps, mixed extremes in each
    n = T.size
    Y = rng.dirichlet(np.full(Ns, 0.3), size=n).T
    Y[rng.random(Y.shape) < 0.25] = 0.0
    Y[rng.random(Y.shape) < 0.10] = 1e-30
    Y[rng.integers(0, Ns, n // 3), np.arange(0, n, 3)[: n // 3]] += 5.0  # one dominant species at every third point
    Y /= Y.sum(axis=0)
    st = dict(T=T, p=p, Y=np.ascontiguousarray(Y))
    gpu, ref = parity.run_gpu(gm, st), parity.run_oracle(om, st)
    for key in ("cp", "h", "mu", "lam", "rhoD", "omega", "qdot"):
        assert np.all(np.isfinite(gpu[key])) and np.all(np.isfinite(ref[key])), key
    parity.assert_parity(gpu, ref, f"{name} extreme states")


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_repeated_launches_are_bit_identical(binding, oracle_mod, name):
    """The kernels use no atomics and a fixed summation order: three launches over the same inputs (enough points
    for every SM to hold its full complement of blocks, so that staging buffers and shared rows are reused under
    load) must agree bit for bit.  A shared-memory race or a read past a staged block would show up here."""
    desc, gm, om = _mech_pair(binding, oracle_mod, name)
    n = 148 * 64 * 6 + 37
    st = wl.make_state(name, n=n, total=n)
    first = parity.run_gpu(gm, st)
    for _ in range(2):
        again = parity.run_gpu(gm, st)
        for key, v in first.items():
            assert np.array_equal(v, again[key]), f"{name}: {key} differs between launches"
