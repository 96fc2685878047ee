"""net_integrate_static: the entry point for callers that cannot allocate device memory.

Some programs that embed this library may not call cudaMalloc once they are running: a hydro
code whose own pool allocator has taken all of HBM, a time loop inside a region where the CUDA
runtime forbids allocation, a driver that must account for every byte before it starts.
net_integrate's only scratch -- the counting sort that launches the hottest zones first -- is
reserved with cudaMalloc by net_create / net_reserve; net_integrate_static keeps the same
scratch in a fixed 264 KB array inside libkinnet.so (include/kinnet.h, NET_STATIC_MAX_ZONES =
65536 zones per call) and allocates nothing.

What is checked here, through the C ABI, against the existing path (net_integrate):
  - two calls in a row on the same stream (the array keeps the first call's contents: the
    second call must not be disturbed by them) return net_integrate's abundances, final dt,
    step counts and status words.  The launch order decides when a zone runs, never what it
    computes (tests/test_gpu_parity.py::test_launch_order_changes_nothing_but_the_schedule), so
    the comparison is bit for bit -- tighter than the 1e-6 adaptive tolerance of the parity
    tests, which is asserted as well so that a failure says how far off it is;
  - a second, smaller batch right behind a larger one (stale order entries beyond the new
    batch must not be read);
  - a batch beyond the limit is refused with a message that names the limit, and nothing runs.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and
a failure here must not hide the parity tests.  It builds its own net_t and inputs, so it passes
alone in a fresh process (where its first call also performs the per-device address lookup) and
after the rest of the suite.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_1409_5826_b200 as K  # noqa: E402
from gen import build_config  # noqa: E402

DEV = "cuda:0"
ADAPT_TOL = 1e-6  # BASELINE.json north_star: adaptive dt, mass fractions above 1e-12
X_MIN = 1e-12


def _dev(a, dtype=torch.float64):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).to(DEV).contiguous()


def _run(call, c, lo, hi):
    """One call of `call` (a bound Net method) on zones [lo, hi) of config c; host copies."""
    z = hi - lo
    T9, rho, Y = _dev(c["T9"][lo:hi]), _dev(c["rho"][lo:hi]), _dev(c["Y0"][lo:hi])
    dt = torch.zeros(z, dtype=torch.float64, device=DEV)
    steps = torch.zeros(z, dtype=torch.int32, device=DEV)
    status = torch.full((z,), -1, dtype=torch.int32, device=DEV)
    call(z, T9, rho, Y, c["t_hydro"], dt, steps, status)
    torch.cuda.synchronize()
    return dict(Y=Y.cpu().numpy(), dt=dt.cpu().numpy(), n_steps=steps.cpu().numpy(),
                status=status.cpu().numpy())


def _same(got, want, A, label):
    m = want["Y"] * A > X_MIN
    err = float(np.abs(got["Y"][m] / want["Y"][m] - 1).max())
    assert err <= ADAPT_TOL, (label, err)
    assert (np.abs(got["n_steps"] - want["n_steps"]) <= np.maximum(1, want["n_steps"] // 100)).all(), label
    for key in ("Y", "dt", "n_steps", "status"):  # and in fact bit for bit
        assert np.array_equal(got[key], want[key]), (label, key)
    assert (got["status"] == 0).all(), label


def test_static_entry_point_matches_net_integrate_twice_in_a_row(hub150):
    z = 2048  # several waves of the GPU, step counts spread over two decades: the order matters
    c = build_config(4, zones=z)
    kn = K.Net(hub150)
    want = _run(kn.net_integrate, c, 0, z)
    first = _run(kn.net_integrate_static, c, 0, z)
    second = _run(kn.net_integrate_static, c, 0, z)
    _same(first, want, hub150.A, "first call")
    _same(second, want, hub150.A, "second call")
    assert want["n_steps"].max() > 20 * want["n_steps"].min()
    # a shorter, different batch behind it: only its own 700 order entries may be used
    want_part = _run(kn.net_integrate, c, 1000, 1700)
    part = _run(kn.net_integrate_static, c, 1000, 1700)
    _same(part, want_part, hub150.A, "shorter batch after a longer one")
    # a second net_t (other kernel family) shares the same array
    kg = K.Net(hub150, K.NetParams(kernel=1))
    _same(_run(kg.net_integrate_static, c, 0, 1024), _run(kg.net_integrate, c, 0, 1024), hub150.A,
          "generic kernel")


def test_static_entry_point_refuses_batches_beyond_its_array(g16):
    kn = K.Net(g16)
    kn.net_integrate_static(0, None, None, None, 1e-9)  # set-up call: legal, launches nothing
    z = K.NET_STATIC_MAX_ZONES + 1
    Y = torch.full((4, g16.n_species), 0.25, dtype=torch.float64, device=DEV)  # never touched
    before = Y.clone()
    with pytest.raises(K.KinnetError) as e:
        kn.net_integrate_static(z, Y, Y, Y, 1e-9)
    assert e.value.code == K.NET_EINVAL
    assert "NET_STATIC_MAX_ZONES" in str(e.value) and str(K.NET_STATIC_MAX_ZONES) in str(e.value)
    torch.cuda.synchronize()
    assert torch.equal(Y, before)
    # the limit itself is accepted
    z = K.NET_STATIC_MAX_ZONES
    rng = np.random.default_rng(65536)
    c1 = build_config(1)
    T9, rho = rng.uniform(1, 10, z), 10 ** rng.uniform(7, 9.5, z)
    c = dict(T9=T9, rho=rho, Y0=np.repeat(c1["Y0"], z, axis=0), t_hydro=1e-9)
    got, want = _run(kn.net_integrate_static, c, 0, z), _run(kn.net_integrate, c, 0, z)
    for key in ("Y", "dt", "n_steps", "status"):
        assert np.array_equal(got[key], want[key]), key
