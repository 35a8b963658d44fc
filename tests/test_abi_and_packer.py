"""CPU-only checks of the boundary and the host logic: libcrf.so loads and exports every symbol
include/crf.h declares (no compute calls without a GPU), the ctypes mirror of ``crf_tables``
has the header's field order, and the packer's re-layout is right (checked against the
description, independently of any kernel)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2409_06404_b200 import binding, build, packer
from paper_2409_06404_b200 import workloads as wl
from tests.helpers import rxn, tiny_mech

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "crf.h")
HEADER_DIAG = os.path.join(ROOT, "include", "crf_diag.h")


@pytest.fixture(scope="module")
def lib_path():
    return build.build()


def _declared_functions(path=HEADER):
    src = open(path).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(crf_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib_path):
    names = _declared_functions()
    assert {"crf_mech_create", "crf_thermo", "crf_production_rates", "crf_mix_transport"} <= set(names)
    L = C.CDLL(lib_path)
    for nm in names:
        assert hasattr(L, nm), f"libcrf.so does not export {nm}"
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS and include/crf.h disagree"
    diag = _declared_functions(HEADER_DIAG)
    for nm in diag:
        assert hasattr(L, nm), f"libcrf.so does not export {nm} (crf_diag.h)"
    assert sorted(binding.EXPORTS_DIAG) == diag, "binding.EXPORTS_DIAG and include/crf_diag.h disagree"
    # the method header holds the method only: no probe, counter or schedule dump
    assert not {"crf_fp64_probe", "crf_launch_count", "crf_transport_schedule"} & set(names)


def test_plan_structs_mirror_header():
    src = re.sub(r"/\*.*?\*/", "", open(HEADER_DIAG).read(), flags=re.S)
    for cname, mirror in (("crf_plan_options", binding.PlanOptions), ("crf_plan_info", binding.PlanInfo)):
        body = re.search(r"typedef struct %s \{(.*?)\} %s;" % (cname, cname), src, flags=re.S).group(1)
        fields = []
        for decl in body.split(";"):
            decl = decl.strip()
            if decl:
                fields += [w.strip(",").split("[")[0] for w in decl.split()[1:]]
        assert fields == [f[0] for f in mirror._fields_], cname


def test_no_environment_tuning_in_the_library():
    """Kernel plans are chosen from the mechanism or requested through crf_plan_options: libcrf.so reads no
    environment variable and carries no work-skipping switch."""
    csrc = os.path.join(ROOT, "paper_2409_06404_b200", "csrc")
    for f in os.listdir(csrc):
        text = open(os.path.join(csrc, f)).read()
        assert "getenv" not in text and "dbg_skip" not in text and "_SKIP" not in text, f


def test_argument_errors_need_no_gpu(lib_path):
    L = binding.lib()
    assert L.crf_mech_create(None, None) == -1
    assert b"null" in L.crf_last_error()
    assert L.crf_mech_num_species(None) == -1
    assert L.crf_thermo(None, None, None, None, 4, None, None) == -1
    assert L.crf_launch_count() == 0
    t = packer.pack(wl.make_mechanism("C1")).as_struct()
    t.version = 99
    h = C.c_void_p()
    assert L.crf_mech_create(C.byref(t), C.byref(h)) == -1 and b"version" in L.crf_last_error()
    # plan options are checked before anything touches a device
    t = packer.pack(wl.make_mechanism("C1")).as_struct()
    for field, bad, word in (("transport_TS", 6, b"transport_TS"), ("thermo_sets", 3, b"thermo_sets"), ("reserved", None, b"reserved")):
        o = binding.PlanOptions()
        if field == "reserved":
            o.reserved[0] = 1
        else:
            setattr(o, field, bad)
        assert L.crf_mech_create_ex(C.byref(t), C.byref(o), C.byref(h)) == -1 and word in L.crf_last_error(), field
    assert L.crf_step_host_static(None, None, None, None, 1, None, None, None, None, None, None, None) == -1
    assert L.crf_step_host_static_max_points(None) == -1


def test_tables_struct_mirrors_header():
    src = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)
    body = re.search(r"typedef struct crf_tables \{(.*?)\} crf_tables;", src, flags=re.S).group(1)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        names = decl.replace("*", " ").split()
        first = next(i for i, w in enumerate(names) if w not in ("const", "int32_t", "int16_t", "double"))
        fields += [w.strip(",") for w in names[first:]]
    assert fields == [f[0] for f in packer.CrfTables._fields_]


def test_packer_layout_and_units():
    m = wl.make_mechanism("C4")
    t = packer.pack(m)
    a = t.arrays
    ns, nr = t.Ns, t.Nr
    assert (ns, nr, t.N3, t.Nt) == (53, 325, 40, 25)
    rx = [m["reactions"][i] for i in t.order]
    kinds = [r["type"] for r in rx]
    ne = nr - t.N3 - t.Nt
    assert kinds == ["elementary"] * ne + ["three_body"] * t.N3 + ["falloff"] * t.Nt
    assert a["nasa_lo"].shape == (7, ns) and np.array_equal(a["nasa_lo"][:, 5], m["nasa_lo"][5])
    assert a["reac"].dtype == np.int16 and a["reac"].shape == (3, nr)
    for i in (0, ne, ne + t.N3, nr - 1):
        r = rx[i]
        molecules = sum(nu for _, nu in r["reactants"])
        third = 1 if r["type"] == "three_body" else 0
        # 1 cm^3/mol = 1e-3 m^3/kmol
        assert np.isclose(a["lnA"][i], np.log(r["A"] * 1e-3 ** (molecules + third - 1)), rtol=1e-14)
        assert np.isclose(a["Ea_R"][i] * 8314.46261815324, r["Ea"] * 1e6, rtol=1e-14)
        listed = sorted(k for k in a["reac"][:, i] if k >= 0)
        assert listed == sorted(k for k, nu in r["reactants"] for _ in range(nu))
    # CSR efficiencies: efficiency - 1, rows in sorted-reaction order
    for row in range(t.N3 + t.Nt):
        r = rx[ne + row]
        lo, hi = a["eff_ptr"][row], a["eff_ptr"][row + 1]
        got = dict(zip(a["eff_idx"][lo:hi].tolist(), (a["eff_val"][lo:hi] + 1.0).tolist()))
        want = {int(k): v for k, v in r["eff"].items() if v != 1.0}
        assert got.keys() == want.keys() and all(np.isclose(got[k], want[k], rtol=1e-15) for k in want)
    # falloff low-pressure limit carries one order more
    r = rx[nr - 1]
    molecules = sum(nu for _, nu in r["reactants"])
    assert np.isclose(a["lnA0"][-1], np.log(r["troe"]["A0"] * 1e-3 ** molecules), rtol=1e-14)
    # pair table: upper triangle including the diagonal, pair (j<=k) at j*Ns - j(j-1)/2 + (k-j)
    D = np.asarray(m["D_fit"])
    assert a["D_c"].shape == (4, ns * (ns + 1) // 2)
    for j, k in ((0, 0), (0, ns - 1), (7, 7), (7, 30), (30, 7), (ns - 1, ns - 1)):
        assert np.array_equal(a["D_c"][:, packer.pair_index(j, k, ns)], D[j, k])


def test_packer_rejects_bad_input():
    W = [2.0, 32.0, 18.0]
    with pytest.raises(ValueError):
        packer.pack(tiny_mech(W, [rxn([(0, 2), (1, 2)], [(2, 1)])]))        # four reactant molecules
    with pytest.raises(ValueError):
        packer.pack(tiny_mech(W, [rxn([(0, 1)], [(2, 1)], A=-1.0)]))         # lnA undefined
    with pytest.raises(ValueError):
        packer.pack(tiny_mech(W, [rxn([(0, 1.5)], [(2, 1)])]))               # fractional coefficient
    m = tiny_mech(W, [])
    m["D_fit"] = np.array(m["D_fit"])
    m["D_fit"][0, 1, 0] += 1.0
    with pytest.raises(ValueError):
        packer.pack(m)                                                       # asymmetric D_jk


def test_generator_matches_config_recipes():
    for name, cfg in wl.CONFIGS.items():
        m = wl.make_mechanism(name)
        kinds = [r["type"] for r in m["reactions"]]
        assert len(m["W"]) == cfg["Ns"] and len(kinds) == cfg["Nr"]
        assert kinds.count("three_body") == cfg["N3"] and kinds.count("falloff") == cfg["Nt"]
        comp = m["comp"]
        for r in m["reactions"]:  # atom balance of every reaction
            lhs = sum(nu * comp[:, k] for k, nu in r["reactants"])
            rhs = sum(nu * comp[:, k] for k, nu in r["products"])
            assert np.array_equal(lhs, rhs)
        st = wl.make_state(name, n=1024, total=1024)
        assert st["Y"].shape == (cfg["Ns"], 1024) and np.allclose(st["Y"].sum(axis=0), 1.0, atol=1e-14)
        assert st["Y"].min() > 0 and st["T"].min() > 250 and st["T"].max() < 2700


@pytest.mark.parametrize("nb", list(range(1, 18)) + [31, 32])
@pytest.mark.parametrize("W", [1, 2, 4, 8])
def test_transport_tile_schedule(lib_path, nb, W):
    """Host logic of the tiled transport kernel (no GPU): the round-robin schedule must visit every unordered pair
    of species blocks and every diagonal block exactly once, a round must hold at most W tiles, and the tiles of a
    round must touch pairwise disjoint blocks (that is what lets the warps update S without atomics)."""
    L = binding.lib()
    L.crf_transport_schedule.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_int32), C.c_int]
    total = nb * (nb - 1) // 2 + nb
    buf = (C.c_int32 * (4 * total))()
    assert L.crf_transport_schedule(nb, W, buf, total) == total
    tiles = np.frombuffer(buf, dtype=np.int32).reshape(total, 4)
    seen = set()
    for rd in np.unique(tiles[:, 0]):
        t = tiles[tiles[:, 0] == rd]
        assert len(t) <= W
        blocks = []
        for _, kind, jb, kb in t:
            assert 0 <= jb <= kb < nb and kind == (2 if jb == kb else 1)
            blocks += [jb] if jb == kb else [jb, kb]
            assert (jb, kb) not in seen
            seen.add((jb, kb))
        assert len(blocks) == len(set(blocks)), f"round {rd} touches a block twice"
    assert len(seen) == total
    assert L.crf_transport_schedule(0, W, None, 0) == -1 and L.crf_transport_schedule(nb, 3 * W + 9, None, 0) == -1
