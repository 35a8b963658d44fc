"""crf_step_host_static: the host-buffer call whose device staging is a static array inside libcrf.so (no cudaMalloc in
the call).  Collected last on purpose (the suite runs with ``pytest -x``): a failure here hides no other test.

The new entry point is checked against the existing path (crf_step_host), on two calls in a row with different inputs
(the shared array keeps the first call's contents; the second call must not see them), for a small and a large
mechanism, and its size limit is checked to be an error, not a fault."""
import numpy as np
import pytest
import torch

from paper_2409_06404_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu

KEYS = ("cp", "h", "omega", "qdot", "mu", "lam", "rhoD")


@pytest.fixture(scope="module")
def binding():
    from paper_2409_06404_b200 import binding as b
    b.lib()
    return b


def _empty_outputs(Ns, n):
    mk = lambda *s: torch.full(s, float("nan"), dtype=torch.float64)  # noqa: E731
    return dict(cp=mk(n), h=mk(n), omega=mk(Ns, n), qdot=mk(n), mu=mk(n), lam=mk(n), rhoD=mk(Ns, n))


@pytest.mark.parametrize("name,n1,n2", [("C1", 4099, 777), ("C5", 2051, 5808)])
def test_static_scratch_matches_step_host_on_two_calls(binding, oracle_mod, name, n1, n2):
    desc = wl.make_mechanism(name)
    gm = binding.Mechanism(desc)
    om = oracle_mod.Oracle(desc)
    assert n2 <= gm.step_host_static_max_points()
    for call, n in enumerate((n1, n2)):  # two calls in a row on the shared array: different sizes and states
        st = wl.make_state(name, n=n, offset=50000 * call, total=1 << 20)
        host = {k: torch.from_numpy(v) for k, v in st.items()}
        ref = gm.step_host(host["T"], host["p"], host["Y"])  # the existing path (allocates its pipeline buffers)
        out = gm.step_host_static(host["T"], host["p"], host["Y"], _empty_outputs(gm.Ns, n))
        # against the existing path, within the tolerance of the parity tests (tests/parity.py: the per-output scales of
        # DESIGN.md section 5, taken from the oracle on a prefix of the batch) ...
        m = min(n, 256)
        sub = {k: np.ascontiguousarray(v[..., :m]) for k, v in st.items()}
        scales = parity.run_oracle(om, sub)
        exp = dict(scales)
        exp.update({k: ref[k].numpy()[..., :m] for k in KEYS})
        parity.assert_parity({k: out[k].numpy()[..., :m] for k in KEYS}, exp, f"step_host_static vs step_host, call {call}")
        # ... and against the oracle itself
        parity.assert_parity({k: out[k].numpy()[..., :m] for k in KEYS}, scales, f"step_host_static vs oracle, call {call}")
        # the two paths run the same kernels on the same batch (n <= one pipeline chunk): the values agree bit for bit
        for k in KEYS:
            assert torch.equal(out[k], ref[k]), (k, call)


def test_static_scratch_output_groups_and_limit(binding):  # noqa: C901
    desc = wl.make_mechanism("C3")
    gm = binding.Mechanism(desc)
    nmax = gm.step_host_static_max_points()
    assert nmax == 29956  # (7 ceil32(n) + 3 ceil32(21 n) <= 2 Mi doubles)
    n = 1000
    st = wl.make_state("C3", n=n, total=n)
    host = {k: torch.from_numpy(v) for k, v in st.items()}
    ref = gm.step_host(host["T"], host["p"], host["Y"])
    part = dict(omega=torch.empty(gm.Ns, n, dtype=torch.float64), qdot=torch.empty(n, dtype=torch.float64))
    gm.step_host_static(host["T"], host["p"], host["Y"], part)
    assert torch.equal(part["omega"], ref["omega"]) and torch.equal(part["qdot"], ref["qdot"])
    with pytest.raises(binding.CrfError, match="together"):
        gm.step_host_static(host["T"], host["p"], host["Y"], dict(omega=part["omega"]))
    # beyond the static array: a clear error, nothing launched
    big = nmax + 1
    stb = wl.make_state("C3", n=big, total=big)
    hb = {k: torch.from_numpy(v) for k, v in stb.items()}
    before = binding.launch_count()
    with pytest.raises(binding.CrfError, match="static scratch"):
        gm.step_host_static(hb["T"], hb["p"], hb["Y"], _empty_outputs(gm.Ns, big))
    assert binding.launch_count() == before
    # exactly at the limit it runs
    stm = {k: np.ascontiguousarray(v[..., :nmax]) for k, v in stb.items()}
    hm = {k: torch.from_numpy(v) for k, v in stm.items()}
    out = gm.step_host_static(hm["T"], hm["p"], hm["Y"], _empty_outputs(gm.Ns, nmax))
    refm = gm.step_host(hm["T"], hm["p"], hm["Y"])
    for k in KEYS:
        assert torch.equal(out[k], refm[k]), k
