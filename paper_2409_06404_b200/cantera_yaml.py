"""Cantera-format YAML -> mechanism description.

The paper generates its kernels from "a combustion model expressed in Cantera format".  This module
reads the subset of that format the hot path needs and returns the same plain description dict that
``workloads.make_mechanism`` returns (the input of ``packer.pack`` and of the oracle's loader): host-side data
handling only, none of the method's arithmetic.  Cantera itself is not required (and not installed here).

What is read
    units         ``length`` (m | cm | mm), ``quantity`` (mol | kmol), ``activation-energy`` (cal/mol, kcal/mol, J/mol,
                  kJ/mol, J/kmol, K); Cantera's defaults (m, kmol, J/kmol) when the block or a key is missing.  Rate
                  parameters must be plain numbers in those units (strings with inline units are rejected).
    species       ``composition``; ``thermo`` with ``model: NASA7``, one or two temperature ranges.
    reactions     ``equation`` with ``<=>`` (or ``=``), integer coefficients written ``2 OH`` or ``OH + OH``, at most
                  three species slots per side, ``+ M`` / ``(+M)`` / ``(+ M)`` third bodies;
                  ``rate-constant {A, b, Ea}``; ``type: three-body`` with ``efficiencies``; ``type: falloff`` with
                  ``low-P-rate-constant``, ``high-P-rate-constant``, ``Troe {A, T3, T1[, T2]}`` (no Troe block = the
                  Lindemann form) and ``efficiencies``; ``duplicate``.
What is not
    Irreversible reactions (``=>``): every reaction of the tables is reversible (include/crf.h); pressure-dependent
    Arrhenius, Chebyshev, SRI, negative pre-exponential factors, non-integer or > 2 stoichiometric coefficients,
    explicit third-body colliders such as ``(+ H2O)``.  Each raises ``ValueError`` naming the reaction.
Transport
    Cantera YAML carries Lennard-Jones parameters, not the CK-style cubic fits in ln T this path evaluates (SURVEY 8(c)
    step 10; producing them needs collision-integral tables and a fitting step, which is Cantera's own
    pre-processing).  They come from a side table: the top-level extension key ``crf-transport-fits`` of the same
    file, or the ``transport_fits`` argument, with
        species:           {name: {mu: [c0..c3], lambda: [c0..c3]}}     ln(mu / Pa s), ln(lambda / (W/m/K)) cubics in ln T
        binary-diffusion:  {"A B": [c0..c3]}                             ln(D / (m^2/s)) at p_ref, every unordered pair
                                                                         and every "A A"
"""
from __future__ import annotations

import re

import numpy as np
import yaml

ATOMIC_MASS = {"H": 1.008, "D": 2.014, "He": 4.002602, "C": 12.011, "N": 14.007, "O": 15.999, "F": 18.998403,
               "Ne": 20.1797, "Si": 28.085, "S": 32.06, "Cl": 35.45, "Ar": 39.948, "Kr": 83.798, "Xe": 131.293}
P_REF = 101325.0
R_KJ = 8.31446261815324e-3   # kJ/(mol K)
CAL = 4.184                  # J per thermochemical calorie

_LENGTH_CM = {"m": 100.0, "cm": 1.0, "mm": 0.1}
_QUANTITY_MOL = {"mol": 1.0, "kmol": 1000.0, "gmol": 1.0}
_EA_TO_KJ_PER_MOL = {"cal/mol": CAL * 1e-3, "kcal/mol": CAL, "J/mol": 1e-3, "kJ/mol": 1.0, "J/kmol": 1e-6,
                     "K": R_KJ}


def _num(x, what):
    if isinstance(x, bool) or not isinstance(x, (int, float)):
        raise ValueError(f"{what}: expected a plain number in the units of the 'units' block, got {x!r}")
    return float(x)


class _Units:
    def __init__(self, block):
        block = block or {}
        try:
            self.cm = _LENGTH_CM[block.get("length", "m")]
            self.mol = _QUANTITY_MOL[block.get("quantity", "kmol")]
            self.ea = _EA_TO_KJ_PER_MOL[block.get("activation-energy", "J/kmol")]
        except KeyError as err:
            raise ValueError(f"units: unsupported unit {err}") from None
        if block.get("time", "s") != "s":
            raise ValueError("units: time must be s")

    def A_to_cgs(self, A, order):
        """(length^3/quantity)^(order-1)/s -> (cm^3/mol)^(order-1)/s"""
        return A * (self.cm ** 3 / self.mol) ** (order - 1)


def _parse_side(text, index, eq):
    """'2 OH + H2O' -> ([(k, nu), ...], has_M) with repeated species merged."""
    counts, has_m = {}, False
    for term in text.split(" + "):
        term = term.strip()
        if not term:
            raise ValueError(f"reaction '{eq}': empty term")
        if term == "M":
            has_m = True
            continue
        m = re.fullmatch(r"(\d+(?:\.\d+)?)\s+(\S+)", term)
        nu, name = (float(m.group(1)), m.group(2)) if m else (1.0, term)
        if nu != int(nu):
            raise ValueError(f"reaction '{eq}': non-integer stoichiometric coefficient {nu}")
        if name not in index:
            raise ValueError(f"reaction '{eq}': unknown species '{name}'")
        counts[index[name]] = counts.get(index[name], 0) + int(nu)
    for k, nu in counts.items():
        if nu > 2:
            raise ValueError(f"reaction '{eq}': stoichiometric coefficient {nu} > 2 is not supported")
    if sum(counts.values()) > 3:
        raise ValueError(f"reaction '{eq}': more than three species slots on one side")
    return [(k, nu) for k, nu in counts.items()], has_m


def _parse_equation(eq, index):
    if "<=>" in eq:
        lhs, rhs = eq.split("<=>")
    elif "=>" in eq:
        raise ValueError(f"reaction '{eq}': irreversible reactions are not supported (every reaction of the tables "
                         "is reversible)")
    elif " = " in eq:
        lhs, rhs = eq.split(" = ")
    else:
        raise ValueError(f"reaction '{eq}': no '<=>'")
    falloff = []
    for side in (lhs, rhs):
        m = re.search(r"\(\s*\+\s*(\S+?)\s*\)", side)
        falloff.append(m.group(1) if m else None)
    if falloff[0] != falloff[1]:
        raise ValueError(f"reaction '{eq}': '(+M)' must appear on both sides")
    if falloff[0] not in (None, "M"):
        raise ValueError(f"reaction '{eq}': explicit falloff collider '(+{falloff[0]})' is not supported")
    strip = lambda s: re.sub(r"\(\s*\+\s*\S+?\s*\)", "", s)  # noqa: E731
    reac, m_l = _parse_side(strip(lhs), index, eq)
    prod, m_r = _parse_side(strip(rhs), index, eq)
    if m_l != m_r:
        raise ValueError(f"reaction '{eq}': '+ M' must appear on both sides")
    if not reac or not prod:
        raise ValueError(f"reaction '{eq}': a side without species")
    return reac, prod, m_l, falloff[0] is not None


def _arrhenius(block, units, order, what):
    if not isinstance(block, dict):
        raise ValueError(f"{what}: expected a mapping {{A, b, Ea}}")
    A = _num(block.get("A"), what + " A")
    if A <= 0.0:
        raise ValueError(f"{what}: pre-exponential factors must be positive")
    return units.A_to_cgs(A, order), _num(block.get("b", 0.0), what + " b"), _num(block.get("Ea", 0.0), what + " Ea") * units.ea


def _efficiencies(block, index, eq):
    out = {}
    for name, e in (block or {}).items():
        if name not in index:
            raise ValueError(f"reaction '{eq}': efficiency for unknown species '{name}'")
        out[index[name]] = _num(e, f"reaction '{eq}' efficiency")
    return out


def _fits(doc, transport_fits, names):
    src = transport_fits if transport_fits is not None else doc.get("crf-transport-fits")
    if src is None:
        raise ValueError("no transport fits: Cantera YAML holds Lennard-Jones parameters, not the cubic fits in ln T this "
                         "path evaluates; pass transport_fits= or add the 'crf-transport-fits' extension key")
    if isinstance(src, str):
        with open(src) as f:
            src = yaml.safe_load(f)
    ns = len(names)
    mu, lam, D = np.empty((ns, 4)), np.empty((ns, 4)), np.empty((ns, ns, 4))

    def four(v, what):
        v = [float(x) for x in v]
        if len(v) != 4:
            raise ValueError(f"transport fits: {what} needs four coefficients")
        return v
    for k, nm in enumerate(names):
        try:
            mu[k] = four(src["species"][nm]["mu"], f"mu of {nm}")
            lam[k] = four(src["species"][nm]["lambda"], f"lambda of {nm}")
        except KeyError:
            raise ValueError(f"transport fits: no mu/lambda fit for species '{nm}'") from None
    pairs = {tuple(sorted(key.split())): four(v, key) for key, v in src.get("binary-diffusion", {}).items()}
    for j, a in enumerate(names):
        for k, b in enumerate(names):
            key = tuple(sorted((a, b)))
            if key not in pairs:
                raise ValueError(f"transport fits: no binary-diffusion fit for the pair '{a} {b}'")
            D[j, k] = pairs[key]
    return mu, lam, D


def load(source, transport_fits=None, phase=None) -> dict:
    """``source``: path of a YAML file or YAML text.  Returns the mechanism description (see ``workloads``)."""
    if "\n" not in source and not source.lstrip().startswith(("{", "units", "phases", "species")):
        with open(source) as f:
            doc = yaml.safe_load(f)
    else:
        doc = yaml.safe_load(source)
    units = _Units(doc.get("units"))
    phases = doc.get("phases") or [{}]
    ph = next((p for p in phases if phase is None or p.get("name") == phase), None)
    if ph is None:
        raise ValueError(f"no phase named '{phase}'")
    species_nodes = {s["name"]: s for s in doc.get("species", [])}
    listed = ph.get("species")
    names = list(species_nodes) if listed in (None, "all") else [str(s) for s in listed]
    for nm in names:
        if nm not in species_nodes:
            raise ValueError(f"species '{nm}' is listed in the phase but not defined")
    index = {nm: k for k, nm in enumerate(names)}
    ns = len(names)
    elements = list(ph.get("elements") or sorted({e for nm in names for e in species_nodes[nm]["composition"]}))
    comp = np.zeros((len(elements), ns), dtype=np.int64)
    tmid, lo, hi = np.empty(ns), np.empty((ns, 7)), np.empty((ns, 7))
    for k, nm in enumerate(names):
        node = species_nodes[nm]
        for e, c in node["composition"].items():
            if e not in elements or e not in ATOMIC_MASS:
                raise ValueError(f"species '{nm}': unknown element '{e}'")
            if c != int(c):
                raise ValueError(f"species '{nm}': non-integer composition")
            comp[elements.index(e), k] = int(c)
        th = node.get("thermo", {})
        if th.get("model") != "NASA7":
            raise ValueError(f"species '{nm}': thermo model must be NASA7")
        tr, data = [float(x) for x in th["temperature-ranges"]], th["data"]
        if len(tr) == 3 and len(data) == 2:
            tmid[k], lo[k], hi[k] = tr[1], data[0], data[1]
        elif len(tr) == 2 and len(data) == 1:
            tmid[k], lo[k], hi[k] = tr[1], data[0], data[0]
        else:
            raise ValueError(f"species '{nm}': NASA7 needs one or two temperature ranges")
    W = comp.T.astype(float) @ np.array([ATOMIC_MASS[e] for e in elements])

    reactions = []
    for node in doc.get("reactions", []):
        eq = str(node["equation"])
        reac, prod, has_m, is_falloff = _parse_equation(eq, index)
        typ = node.get("type", "three-body" if has_m else "elementary")
        molecules = sum(nu for _, nu in reac)
        if typ == "elementary" and not has_m and not is_falloff:
            A, b, Ea = _arrhenius(node.get("rate-constant"), units, molecules, f"reaction '{eq}'")
            r = dict(reactants=reac, products=prod, type="elementary", A=A, beta=b, Ea=Ea)
        elif typ == "three-body" and has_m and not is_falloff:
            A, b, Ea = _arrhenius(node.get("rate-constant"), units, molecules + 1, f"reaction '{eq}'")
            r = dict(reactants=reac, products=prod, type="three_body", A=A, beta=b, Ea=Ea,
                     eff=_efficiencies(node.get("efficiencies"), index, eq))
        elif typ == "falloff" and is_falloff and not has_m:
            A, b, Ea = _arrhenius(node.get("high-P-rate-constant"), units, molecules, f"reaction '{eq}' high-P")
            A0, b0, Ea0 = _arrhenius(node.get("low-P-rate-constant"), units, molecules + 1, f"reaction '{eq}' low-P")
            if "SRI" in node:
                raise ValueError(f"reaction '{eq}': SRI falloff is not supported")
            t = node.get("Troe")
            if t is None:   # Lindemann: F = 1 is the Troe form with alpha = 1 and the three temperatures at infinity
                alpha, T3, T1, T2 = 1.0, 1e300, 1e300, 1e300
            else:
                alpha, T3, T1 = _num(t["A"], "Troe A"), _num(t["T3"], "Troe T3"), _num(t["T1"], "Troe T1")
                T2 = _num(t["T2"], "Troe T2") if "T2" in t else 1e300  # no fourth parameter: the term exp(-T2/T) is 0
            r = dict(reactants=reac, products=prod, type="falloff", A=A, beta=b, Ea=Ea,
                     eff=_efficiencies(node.get("efficiencies"), index, eq),
                     troe=dict(A0=A0, beta0=b0, Ea0=Ea0, alpha=alpha, T3=T3, T1=T1, T2=T2))
        else:
            raise ValueError(f"reaction '{eq}': type '{typ}' is not supported or does not match the equation")
        r["equation"], r["duplicate"] = eq, bool(node.get("duplicate", False))
        bal = sum(nu * comp[:, k] for k, nu in prod) - sum(nu * comp[:, k] for k, nu in reac)
        if np.any(bal != 0):
            raise ValueError(f"reaction '{eq}': atoms are not balanced")
        reactions.append(r)
    mu, lam, D = _fits(doc, transport_fits, names)
    return dict(name=str(ph.get("name", "yaml")), elements=elements, species=names, comp=comp, W=W, nasa_Tmid=tmid,
                nasa_lo=lo, nasa_hi=hi, reactions=reactions, mu_fit=mu, lam_fit=lam, D_fit=D, p_ref=P_REF)
