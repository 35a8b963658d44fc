"""Host-side mechanism packer: mechanism description -> species-major SoA tables (``crf_tables``).

Input is the description dict documented in ``workloads.py`` (cgs-mol Arrhenius data, kJ/mol
activation energies, dense symmetric D_jk fits).  Output is a ``PackedTables`` holding one
contiguous numpy array per coefficient in the layout ``include/crf.h`` documents:

* reactions sorted by type (elementary | third-body | Troe falloff) so that every kernel loop
  is uniform (SURVEY.md §7 "Divergence");
* rate constants in SI-kmol units, as logarithms: ``lnA = ln(A_cgs) - (order-1) ln 1000``
  (1 cm^3/mol = 1e-3 m^3/kmol; order counts the third body, and the low-pressure limit of a
  falloff reaction has one order more than its high-pressure limit), ``Ea_R = Ea / R`` in K;
* stoichiometry as up to three reactant and three product slots (-1 = empty, a species listed
  twice = coefficient 2);
* third-body efficiencies as CSR of (efficiency - 1);
* NASA-7 and transport fits coefficient-major (``[c][k]``), D_jk as the upper triangle
  including the diagonal.

This is product code: it shares nothing with ``oracle/``.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass, field

import numpy as np

R_KJ_PER_MOL_K = 8.31446261815324e-3
TABLES_VERSION = 1
MAX_SLOTS = 3
_TYPE_ORDER = {"elementary": 0, "three_body": 1, "falloff": 2}


class CrfTables(C.Structure):
    """ctypes mirror of ``struct crf_tables`` (include/crf.h)."""
    _fields_ = ([(n, C.c_int32) for n in ("version", "Ns", "Nr", "N3", "Nt", "reserved")]
                + [("p_ref", C.c_double)]
                + [(n, C.c_void_p) for n in
                   ("W", "Tmid", "nasa_lo", "nasa_hi", "lnA", "beta", "Ea_R", "reac", "prod",
                    "eff_ptr", "eff_idx", "eff_val", "lnA0", "beta0", "Ea0_R", "alpha", "T3", "T1", "T2",
                    "mu_c", "lam_c", "D_c")])


@dataclass
class PackedTables:
    Ns: int
    Nr: int
    N3: int
    Nt: int
    p_ref: float
    arrays: dict = field(default_factory=dict)
    order: np.ndarray | None = None  # order[i] = index in the description of packed reaction i

    def as_struct(self) -> CrfTables:
        """The C struct; it borrows the numpy buffers of ``self.arrays`` (keep ``self`` alive)."""
        s = CrfTables(version=TABLES_VERSION, Ns=self.Ns, Nr=self.Nr, N3=self.N3, Nt=self.Nt,
                      reserved=0, p_ref=self.p_ref)
        for name, arr in self.arrays.items():
            setattr(s, name, arr.ctypes.data_as(C.c_void_p))
        return s


def pair_index(j: int, k: int, ns: int) -> int:
    """Index of the unordered pair (j, k) in the upper triangle incl. the diagonal."""
    if j > k:
        j, k = k, j
    return j * ns - j * (j - 1) // 2 + (k - j)


def _slots(side, nr_slot):
    out = []
    for k, nu in side:
        if int(nu) != nu or nu < 1:
            raise ValueError(f"stoichiometric coefficient {nu} is not a positive integer")
        out += [int(k)] * int(nu)
    if not 1 <= len(out) <= nr_slot:
        raise ValueError(f"{len(out)} molecules on one side: the tables hold 1..{nr_slot}")
    return out + [-1] * (nr_slot - len(out))


def pack(mech: dict) -> PackedTables:
    ns = len(mech["W"])
    rx_all = mech["reactions"]
    order = np.array(sorted(range(len(rx_all)), key=lambda i: (_TYPE_ORDER[rx_all[i]["type"]], i)), dtype=np.int64)
    rx = [rx_all[i] for i in order]
    nr = len(rx)
    n3 = sum(r["type"] == "three_body" for r in rx)
    nt = sum(r["type"] == "falloff" for r in rx)
    f64 = lambda a: np.ascontiguousarray(a, dtype=np.float64)  # noqa: E731
    a = {}
    a["W"] = f64(mech["W"])
    a["Tmid"] = f64(mech["nasa_Tmid"])
    a["nasa_lo"] = f64(np.asarray(mech["nasa_lo"], dtype=np.float64).reshape(ns, 7).T)
    a["nasa_hi"] = f64(np.asarray(mech["nasa_hi"], dtype=np.float64).reshape(ns, 7).T)

    ln1000 = np.log(1000.0)
    lnA, beta, Ea_R = np.zeros(nr), np.zeros(nr), np.zeros(nr)
    reac = np.full((MAX_SLOTS, nr), -1, dtype=np.int16)
    prod = np.full((MAX_SLOTS, nr), -1, dtype=np.int16)
    eff_ptr, eff_idx, eff_val = [0], [], []
    troe = {k: [] for k in ("lnA0", "beta0", "Ea0_R", "alpha", "T3", "T1", "T2")}
    for i, r in enumerate(rx):
        rs, ps = _slots(r["reactants"], MAX_SLOTS), _slots(r["products"], MAX_SLOTS)
        for k in rs + ps:
            if k >= ns:
                raise ValueError(f"species index {k} out of range")
        reac[:, i], prod[:, i] = rs, ps
        molecules = sum(k >= 0 for k in rs)
        if r["A"] <= 0.0:
            raise ValueError("pre-exponential factors must be positive (stored as logarithms)")
        third = 1 if r["type"] == "three_body" else 0
        lnA[i] = np.log(r["A"]) - (molecules + third - 1) * ln1000
        beta[i] = r["beta"]
        Ea_R[i] = r["Ea"] / R_KJ_PER_MOL_K
        if r["type"] != "elementary":
            for k, e in sorted(r.get("eff", {}).items()):
                if e != 1.0:
                    eff_idx.append(int(k))
                    eff_val.append(float(e) - 1.0)
            eff_ptr.append(len(eff_idx))
        if r["type"] == "falloff":
            t = r["troe"]
            if t["A0"] <= 0.0:
                raise ValueError("pre-exponential factors must be positive (stored as logarithms)")
            troe["lnA0"].append(np.log(t["A0"]) - molecules * ln1000)
            troe["beta0"].append(t["beta0"])
            troe["Ea0_R"].append(t["Ea0"] / R_KJ_PER_MOL_K)
            for key in ("alpha", "T3", "T1", "T2"):
                troe[key].append(t[key])
    a.update(lnA=lnA, beta=beta, Ea_R=Ea_R, reac=np.ascontiguousarray(reac), prod=np.ascontiguousarray(prod))
    a["eff_ptr"] = np.asarray(eff_ptr, dtype=np.int32)
    a["eff_idx"] = np.asarray(eff_idx if eff_idx else [0], dtype=np.int16)
    a["eff_val"] = f64(eff_val if eff_val else [0.0])
    for key, v in troe.items():
        a[key] = f64(v if v else [0.0])

    a["mu_c"] = f64(np.asarray(mech["mu_fit"], dtype=np.float64).reshape(ns, 4).T)
    a["lam_c"] = f64(np.asarray(mech["lam_fit"], dtype=np.float64).reshape(ns, 4).T)
    D = np.asarray(mech["D_fit"], dtype=np.float64).reshape(ns, ns, 4)
    if not np.array_equal(D, D.transpose(1, 0, 2)):
        raise ValueError("D_fit must be symmetric in the species pair")
    iu = np.triu_indices(ns)
    a["D_c"] = f64(D[iu[0], iu[1]].T)
    return PackedTables(Ns=ns, Nr=nr, N3=n3, Nt=nt, p_ref=float(mech["p_ref"]), arrays=a, order=order)
