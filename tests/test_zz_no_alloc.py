"""tfstat_marginalise_static -- the entry point that allocates nothing (its scratch is a static
__device__ array inside libtfstat.so, include/tfstat.h) -- against tfstat_marginalise, the
existing path with a caller-owned workspace, on two calls in a row that share the scratch (-m gpu).

The file sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not
hide the parity tests.  It passes alone in a fresh process and after the other tests."""
import ctypes as C

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from tests.parity import TOL_2F, TOL_LOGB  # noqa: E402

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    import paper_1805_05652_b200 as p

    p.load_library()
    assert torch.cuda.is_available()
    return p


def _random_map(seed, N_t0, N_tau, flagged):
    """A map like the kernels write: 2F >= 0 with a chi^2_4-like bulk and a few loud cells,
    flagged cells (2F = 0, flag != 0) sprinkled in."""
    g = torch.Generator(device="cuda").manual_seed(seed)
    m = (torch.randn((4, N_t0, N_tau), device="cuda", generator=g) ** 2).sum(0)
    m[torch.rand((N_t0, N_tau), device="cuda", generator=g) < 1e-4] *= 7.0
    f = (torch.rand((N_t0, N_tau), device="cuda", generator=g) < flagged).to(torch.uint8)
    f *= 1 + (torch.rand((N_t0, N_tau), device="cuda", generator=g) < 0.5).to(torch.uint8)
    return torch.where(f != 0, torch.zeros_like(m), m).contiguous(), f.contiguous()


def _same(got, ref):
    assert int(got["n_valid"]) == int(ref["n_valid"])
    assert (int(got["m"]), int(got["n"])) == (int(ref["m"]), int(ref["n"]))
    assert abs(float(got["max2F"]) - float(ref["max2F"])) <= TOL_2F * max(1.0, float(ref["max2F"]))
    if int(ref["n_valid"]):
        assert abs(float(got["logB"]) - float(ref["logB"])) <= TOL_LOGB * max(1.0, abs(float(ref["logB"])))
    else:
        assert float(got["logB"]) == float(ref["logB"]) == -np.inf


def test_marginalise_static_equals_workspace_path_two_calls_in_a_row(pkg):
    """First a large map (every one of the 1184 scratch records is written), then, straight after
    it and into the same scratch, a small one (13 records: stale records of the first call must
    not count), then a map with every cell flagged.  Each against tfstat_marginalise; the caller
    passes inputs and the output, the call allocates nothing."""
    out = torch.empty((1, 5), dtype=torch.int32, device="cuda")
    cases = [(11, 2100, 3001, 0.01, True), (12, 37, 1417, 0.2, True), (13, 5, 7, 0.0, False),
             (14, 64, 64, 2.0, True)]
    for seed, N_t0, N_tau, flagged, with_flags in cases:
        m, f = _random_map(seed, N_t0, N_tau, flagged)
        fl = f if with_flags else None
        ref = pkg.tfstat_marginalise(m, fl).numpy()[0]
        got = pkg.tfstat_marginalise_static(m, fl, out=out).numpy()[0]
        _same(got, ref)
        # the same kernels ran: not only within tolerance but the same bits
        assert got.tobytes() == ref.tobytes()
        if flagged >= 1.0:
            assert int(got["n_valid"]) == 0 and (int(got["m"]), int(got["n"])) == (-1, -1)
    # a repeated call sees the scratch its predecessor left: same answer again
    m, f = _random_map(12, 37, 1417, 0.2)
    a = pkg.tfstat_marginalise_static(m, f).numpy()[0]
    b = pkg.tfstat_marginalise_static(m, f).numpy()[0]
    assert a.tobytes() == b.tobytes()
    _same(a, pkg.tfstat_marginalise(m, f).numpy()[0])


def test_marginalise_static_rejects_what_it_cannot_serve(pkg):
    lib = pkg.load_library()
    m, _ = _random_map(15, 8, 8, 0.0)
    out = torch.empty((1, 5), dtype=torch.int32, device="cuda")
    assert lib.tfstat_marginalise_static_max_cells() == 2**31 - 1
    args = (m.data_ptr(), None)
    # beyond the maximum: refused before anything is launched (the map pointer is never read)
    assert lib.tfstat_marginalise_static(*args, 65536, 32768, out.data_ptr(), None) == -1
    assert lib.tfstat_marginalise_static(*args, 2**31 - 1, 2, out.data_ptr(), None) == -1
    assert lib.tfstat_marginalise_static(*args, 0, 8, out.data_ptr(), None) == -1
    assert lib.tfstat_marginalise_static(None, None, 8, 8, out.data_ptr(), None) == -1
    assert lib.tfstat_marginalise_static(*args, 8, 8, None, None) == -1
    torch.cuda.synchronize()
    # and the entry point still works afterwards
    got = pkg.tfstat_marginalise_static(m, out=out).numpy()[0]
    _same(got, pkg.tfstat_marginalise(m).numpy()[0])
    assert C.sizeof(C.c_size_t) == 8
