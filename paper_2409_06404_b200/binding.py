"""Thin ctypes binding of libcrf.so (include/crf.h).  Argument marshalling only: every step of
the path runs in the CUDA kernels of ``csrc/``.  PyTorch supplies device memory and streams.

There is no CPU fallback: if ``libcrf.so`` is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import packer

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcrf.so")
_lib = None

# include/crf.h (the method) and include/crf_diag.h (plan control, diagnostics)
EXPORTS = ("crf_mech_create", "crf_mech_destroy", "crf_mech_set_stream", "crf_mech_num_species",
           "crf_mech_num_reactions", "crf_thermo", "crf_thermo_species", "crf_production_rates",
           "crf_mix_transport", "crf_rhs_pointwise", "crf_production_rates_pair", "crf_production_rates_jv",
           "crf_production_rates_jv_base",
           "crf_sem_diffusion", "crf_step_host", "crf_step_host_f32", "crf_step_host_static",
           "crf_step_host_static_max_points", "crf_last_error")
EXPORTS_DIAG = ("crf_mech_create_ex", "crf_mech_plan_info", "crf_fp64_probe", "crf_launch_count",
                "crf_transport_schedule")

RATES_KERNELS = {"auto": 0, "generic": 1, "staged": 2, "group": 3, "thread": 4}
TRANSPORT_KERNELS = {"auto": 0, "generic": 1, "small": 2, "tiled": 3}


class PlanOptions(C.Structure):
    """ctypes mirror of ``crf_plan_options`` (include/crf_diag.h)."""
    _fields_ = [(n, C.c_int32) for n in ("rates_kernel", "rates_W", "rates_PPL", "rates_Rc", "transport_kernel",
                                         "transport_W", "transport_PPL", "transport_panel", "rates_tmem", "transport_TS",
                                         "thermo_sets")] \
        + [("reserved", C.c_int32 * 5)]


class PlanInfo(C.Structure):
    """ctypes mirror of ``crf_plan_info`` (include/crf_diag.h)."""
    _fields_ = [(n, C.c_int32) for n in ("rates_kernel", "rates_W", "rates_PPL", "rates_Rc", "rates_chunks",
                                         "rates_stage_bytes", "rates_smem_bytes", "transport_kernel", "transport_W",
                                         "transport_PPL", "transport_nb", "transport_stage_blocks",
                                         "transport_stage_bytes", "transport_smem_bytes", "rates_tmem_cols", "transport_TS",
                                         "thermo_sets")] \
        + [("reserved", C.c_int32 * 5)]


class CrfError(RuntimeError):
    pass


def lib() -> C.CDLL:
    """Loads libcrf.so (built in-tree by ``build.py``); raises if it is not there."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise CrfError(f"{LIB_PATH} not found: run `python -m paper_2409_06404_b200.build` "
                           "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i64, dp = C.c_void_p, C.c_int64, C.c_void_p
        L.crf_mech_create.argtypes = [C.POINTER(packer.CrfTables), C.POINTER(vp)]
        L.crf_mech_create_ex.argtypes = [C.POINTER(packer.CrfTables), C.POINTER(PlanOptions), C.POINTER(vp)]
        L.crf_mech_plan_info.argtypes = [vp, C.POINTER(PlanInfo)]
        L.crf_mech_destroy.argtypes = [vp]
        L.crf_mech_destroy.restype = None
        L.crf_mech_set_stream.argtypes = [vp, vp]
        L.crf_mech_num_species.argtypes = [vp]
        L.crf_mech_num_reactions.argtypes = [vp]
        L.crf_thermo.argtypes = [vp, dp, dp, dp, i64, dp, dp]
        L.crf_thermo_species.argtypes = [vp, dp, i64, dp, dp, dp]
        L.crf_production_rates.argtypes = [vp, dp, dp, dp, i64, dp, dp]
        L.crf_mix_transport.argtypes = [vp, dp, dp, dp, i64, dp, dp, dp]
        L.crf_rhs_pointwise.argtypes = [vp, dp, dp, dp, i64] + [dp] * 10
        L.crf_production_rates_pair.argtypes = [vp] + [dp] * 6 + [i64] + [dp] * 4
        L.crf_production_rates_jv.argtypes = [vp] + [dp] * 6 + [C.c_double, i64] + [dp] * 4
        L.crf_production_rates_jv_base.argtypes = [vp] + [dp] * 6 + [C.c_double, i64] + [dp] * 4
        L.crf_sem_diffusion.argtypes = [vp] + [dp] * 6 + [i64, dp, dp]
        L.crf_step_host.argtypes = [vp, dp, dp, dp, i64] + [dp] * 7
        L.crf_step_host_f32.argtypes = [vp, dp, dp, dp, i64] + [dp] * 7
        L.crf_step_host_static.argtypes = [vp, dp, dp, dp, i64] + [dp] * 7
        L.crf_step_host_static_max_points.argtypes = [vp]
        L.crf_step_host_static_max_points.restype = C.c_int64
        L.crf_fp64_probe.argtypes = [C.c_int, C.POINTER(C.c_double)]
        L.crf_launch_count.restype = C.c_int64
        L.crf_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(code: int):
    if code != 0:
        raise CrfError(f"libcrf error {code}: {lib().crf_last_error().decode()}")


def launch_count() -> int:
    return int(lib().crf_launch_count())


def fp64_probe(iters: int = 4096) -> float:
    """Measured sustained FP64 instructions/s of the current device (crf_fp64_probe)."""
    out = C.c_double()
    _check(lib().crf_fp64_probe(int(iters), C.byref(out)))
    return out.value


def _dev(t: torch.Tensor | None, shape=None):
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise CrfError("expected a contiguous float64 CUDA tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise CrfError(f"expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t.data_ptr()


def _host(t: torch.Tensor, shape):
    if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
        raise CrfError(f"expected a contiguous float64 host tensor of shape {tuple(shape)}")
    return t.data_ptr()


class Mechanism:
    """Device-resident mechanism (``crf_mech``).  ``mech`` is a description dict or PackedTables.
    ``options``: explicit kernel plan (``crf_plan_options``; kernels by name or number), default automatic."""

    def __init__(self, mech, options: dict | None = None):
        self.tables = mech if isinstance(mech, packer.PackedTables) else packer.pack(mech)
        self.Ns, self.Nr = self.tables.Ns, self.tables.Nr
        handle = C.c_void_p()
        struct = self.tables.as_struct()
        if options:
            o = dict(options)
            if isinstance(o.get("rates_kernel"), str):
                o["rates_kernel"] = RATES_KERNELS[o["rates_kernel"]]
            if isinstance(o.get("transport_kernel"), str):
                o["transport_kernel"] = TRANSPORT_KERNELS[o["transport_kernel"]]
            po = PlanOptions(**o)
            _check(lib().crf_mech_create_ex(C.byref(struct), C.byref(po), C.byref(handle)))
        else:
            _check(lib().crf_mech_create(C.byref(struct), C.byref(handle)))
        self._h = handle

    def plan_info(self) -> dict:
        """What this mechanism's calls will run (``crf_mech_plan_info``); kernels by name."""
        info = PlanInfo()
        _check(lib().crf_mech_plan_info(self._h, C.byref(info)))
        d = {n: getattr(info, n) for n, _ in PlanInfo._fields_ if n != "reserved"}
        d["rates_kernel"] = {v: k for k, v in RATES_KERNELS.items()}[d["rates_kernel"]]
        d["transport_kernel"] = {v: k for k, v in TRANSPORT_KERNELS.items()}[d["transport_kernel"]]
        return d

    def close(self):
        if getattr(self, "_h", None):
            lib().crf_mech_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:  # interpreter shutdown: the module's globals (and the library handle) may be gone already
            pass

    def _sync_stream(self):
        _check(lib().crf_mech_set_stream(self._h, C.c_void_p(torch.cuda.current_stream().cuda_stream)))

    def thermo(self, T, p, Y, cp=None, h=None):
        n = T.numel()
        cp = torch.empty_like(T) if cp is None else cp
        h = torch.empty_like(T) if h is None else h
        self._sync_stream()
        _check(lib().crf_thermo(self._h, _dev(T, (n,)), _dev(p), _dev(Y, (self.Ns, n)), n,
                                _dev(cp, (n,)), _dev(h, (n,))))
        return cp, h

    def thermo_species(self, T):
        n = T.numel()
        out = [torch.empty((self.Ns, n), dtype=torch.float64, device=T.device) for _ in range(3)]
        self._sync_stream()
        _check(lib().crf_thermo_species(self._h, _dev(T, (n,)), n, *[_dev(o) for o in out]))
        return tuple(out)

    def production_rates(self, T, p, Y, omega=None, qdot=None):
        n = T.numel()
        omega = torch.empty_like(Y) if omega is None else omega
        qdot = torch.empty_like(T) if qdot is None else qdot
        self._sync_stream()
        _check(lib().crf_production_rates(self._h, _dev(T, (n,)), _dev(p, (n,)), _dev(Y, (self.Ns, n)), n,
                                          _dev(omega, (self.Ns, n)), _dev(qdot, (n,))))
        return omega, qdot

    def mix_transport(self, T, p, Y, mu=None, lam=None, rhoD=None):
        n = T.numel()
        mu = torch.empty_like(T) if mu is None else mu
        lam = torch.empty_like(T) if lam is None else lam
        rhoD = torch.empty_like(Y) if rhoD is None else rhoD
        self._sync_stream()
        _check(lib().crf_mix_transport(self._h, _dev(T, (n,)), _dev(p), _dev(Y, (self.Ns, n)), n,
                                       _dev(mu, (n,)), _dev(lam, (n,)), _dev(rhoD, (self.Ns, n))))
        return mu, lam, rhoD

    def rhs_pointwise(self, T, p, Y, out: dict | None = None, want_cpk: bool = True) -> dict:
        """``crf_rhs_pointwise``: dict(omega, qdot, cp, h, cpk, rho, Wbar, mu, lam, rhoD) of device tensors."""
        n = T.numel()
        if out is None:
            out = {k: torch.empty_like(T) for k in ("qdot", "cp", "h", "rho", "Wbar", "mu", "lam")}
            out.update({k: torch.empty_like(Y) for k in ("omega", "rhoD")})
            out["cpk"] = torch.empty_like(Y) if want_cpk else None
        self._sync_stream()
        _check(lib().crf_rhs_pointwise(
            self._h, _dev(T, (n,)), _dev(p, (n,)), _dev(Y, (self.Ns, n)), n, _dev(out["omega"], (self.Ns, n)),
            _dev(out["qdot"], (n,)), _dev(out["cp"], (n,)), _dev(out["h"], (n,)), _dev(out.get("cpk")),
            _dev(out["rho"], (n,)), _dev(out["Wbar"], (n,)), _dev(out["mu"], (n,)), _dev(out["lam"], (n,)),
            _dev(out["rhoD"], (self.Ns, n))))
        return out

    def production_rates_pair(self, T, p, Y, T2, p2, Y2, out=None):
        """``crf_production_rates_pair``: (omega, qdot, omega2, qdot2)."""
        n = T.numel()
        if out is None:
            out = (torch.empty_like(Y), torch.empty_like(T), torch.empty_like(Y), torch.empty_like(T))
        self._sync_stream()
        _check(lib().crf_production_rates_pair(
            self._h, _dev(T, (n,)), _dev(p, (n,)), _dev(Y, (self.Ns, n)), _dev(T2, (n,)), _dev(p2, (n,)),
            _dev(Y2, (self.Ns, n)), n, _dev(out[0], (self.Ns, n)), _dev(out[1], (n,)), _dev(out[2], (self.Ns, n)),
            _dev(out[3], (n,))))
        return out

    def production_rates_jv(self, T, p, Y, dT, dp, dY, sigma, out=None, base=True):
        """``crf_production_rates_jv``: (omega, qdot, Jomega, Jqdot); omega, qdot are None when ``base`` is False."""
        n = T.numel()
        if out is None:
            out = (torch.empty_like(Y) if base else None, torch.empty_like(T) if base else None,
                   torch.empty_like(Y), torch.empty_like(T))
        self._sync_stream()
        _check(lib().crf_production_rates_jv(
            self._h, _dev(T, (n,)), _dev(p, (n,)), _dev(Y, (self.Ns, n)), _dev(dT, (n,)), _dev(dp),
            _dev(dY, (self.Ns, n)), float(sigma), n, _dev(out[0]), _dev(out[1]), _dev(out[2], (self.Ns, n)),
            _dev(out[3], (n,))))
        return out

    def production_rates_jv_base(self, T, p, Y, dT, dp, dY, sigma, omega, qdot, out=None):
        """``crf_production_rates_jv_base``: (Jomega, Jqdot) against the given base values omega(y), qdot(y) (inputs)."""
        n = T.numel()
        if out is None:
            out = (torch.empty_like(Y), torch.empty_like(T))
        self._sync_stream()
        _check(lib().crf_production_rates_jv_base(
            self._h, _dev(T, (n,)), _dev(p, (n,)), _dev(Y, (self.Ns, n)), _dev(dT, (n,)), _dev(dp),
            _dev(dY, (self.Ns, n)), float(sigma), n, _dev(omega, (self.Ns, n)), _dev(qdot, (n,)),
            _dev(out[0], (self.Ns, n)), _dev(out[1], (n,))))
        return out

    def sem_diffusion(self, h3, T, Wbar, Y, lam, rhoD, dY=None, dT=None):
        """``crf_sem_diffusion``: (dY [Ns, n], dT [n]) on nel = h3.shape[0] order-7 elements, n = 512 nel."""
        nel = h3.shape[0]
        n = 512 * nel
        dY = torch.empty_like(Y) if dY is None else dY
        dT = torch.empty_like(T) if dT is None else dT
        self._sync_stream()
        _check(lib().crf_sem_diffusion(self._h, _dev(h3, (nel, 3)), _dev(T, (n,)), _dev(Wbar, (n,)), _dev(Y, (self.Ns, n)),
                                       _dev(lam, (n,)), _dev(rhoD, (self.Ns, n)), nel, _dev(dY, (self.Ns, n)), _dev(dT, (n,))))
        return dY, dT

    def step_host_static_max_points(self) -> int:
        """Largest batch ``step_host_static`` accepts for this mechanism (``crf_step_host_static_max_points``)."""
        r = int(lib().crf_step_host_static_max_points(self._h))
        if r < 0:
            _check(r)
        return r

    def step_host_static(self, T, p, Y, out: dict) -> dict:
        """``crf_step_host_static``: the whole path with HOST tensors and no allocation in the library: the device staging
        is a 16 MiB array inside libcrf.so, so the batch is limited (``step_host_static_max_points``) and ``out`` (host
        float64 tensors; groups as in ``step_host``) must be given.  Runs on torch's current stream; calls that overlap
        on the GPU race on the shared array."""
        n = T.numel()
        self._sync_stream()
        hp = lambda key, shape: None if out.get(key) is None else _host(out[key], shape)  # noqa: E731
        _check(lib().crf_step_host_static(
            self._h, _host(T, (n,)), _host(p, (n,)), _host(Y, (self.Ns, n)), n,
            hp("cp", (n,)), hp("h", (n,)), hp("omega", (self.Ns, n)), hp("qdot", (n,)), hp("mu", (n,)), hp("lam", (n,)),
            hp("rhoD", (self.Ns, n))))
        return out

    def step_host(self, T, p, Y, out: dict | None = None) -> dict:
        """Whole path with HOST tensors (pinned for full bandwidth); returns host tensors."""
        n = T.numel()
        if out is None:
            mk = lambda *s: torch.empty(s, dtype=torch.float64)  # noqa: E731
            out = dict(cp=mk(n), h=mk(n), omega=mk(self.Ns, n), qdot=mk(n), mu=mk(n), lam=mk(n),
                       rhoD=mk(self.Ns, n))
        f32 = any(v is not None and v.dtype == torch.float32 for v in out.values())

        def hp(key, shape):  # (an output left out of ``out``, or None, is not computed: crf.h)
            if out.get(key) is None:
                return None
            t = out[key]
            if f32:  # float32 outputs: crf_step_host_f32 (double arithmetic, outputs rounded once on the device)
                if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
                    raise CrfError(f"expected a contiguous float32 host tensor of shape {tuple(shape)}")
                return t.data_ptr()
            return _host(t, shape)
        _check((lib().crf_step_host_f32 if f32 else lib().crf_step_host)(
            self._h, _host(T, (n,)), _host(p, (n,)), _host(Y, (self.Ns, n)), n,
            hp("cp", (n,)), hp("h", (n,)), hp("omega", (self.Ns, n)), hp("qdot", (n,)), hp("mu", (n,)), hp("lam", (n,)),
            hp("rhoD", (self.Ns, n))))
        return out
