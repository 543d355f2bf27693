"""opx_prefilter_noalloc: the pre-propagation filter for callers that cannot allocate device memory.

Who that is: code that runs inside somebody else's process -- a Geant4 worker or an experiment-framework plug-in whose
photon buffers come from the framework's memory pool (the pool owns the card; the plug-in is not allowed a cudaMalloc
of its own) -- and worker threads that share one GPU, for which a cudaMalloc / cudaFree is a stall of every other
thread's stream.  They have inputs and outputs but no workspace to hand to opx_prefilter, so the library keeps that
scratch in a fixed array of its own (about 2 MiB per GPU, at most 2^24 photons per call).

What is checked: on two calls in a row through the one shared scratch array -- a large one, then a smaller one that
finds the first call's masks and counts still lying there -- the survivors, their order, their copied bits and the
count are the same bytes opx_prefilter writes with a caller-provided workspace (the filter is integer ranks over
integer masks, so the bar is bit-exact, as in test_gpu_filter.py); and that a call beyond the limit is refused with a
message that names the limit, leaving the outputs alone.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here should not hide the
parity tests.  It builds its own scene and depends on no state of the other tests, so it passes alone in a fresh
process (where its first call is the one that looks up the array's device address) as well as after them."""
import numpy as np
import pytest

import paper_2309_12496_b200 as pkg
import workloads as wl
from paper_2309_12496_b200 import opx

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

KEYS = ("origins", "dirs", "wavelengths", "index")


def _caller_buffers(cap, poison):
    """The caller's own output arrays, filled with a pattern so that entries the call must not touch are recognisable."""
    out = dict(origins=torch.full((cap, 3), poison, dtype=torch.float32, device="cuda"),
               dirs=torch.full((cap, 3), poison, dtype=torch.float32, device="cuda"),
               wavelengths=torch.full((cap,), poison, dtype=torch.float32, device="cuda"),
               index=torch.full((cap,), -7, dtype=torch.int32, device="cuda"),
               n_kept=torch.full((1,), 12345, dtype=torch.int64, device="cuda"))
    return out


def _bytes(out, k):
    torch.cuda.synchronize()
    return {key: out[key][:k].cpu().numpy().view(np.uint32) for key in KEYS}


def test_two_calls_in_a_row_match_the_workspace_path():
    w = wl.make_config("C3", n=600_000)
    sc = w.scene
    gs = pkg.Scene(sc).build()
    fac = [sc.info["m_det"], sc.info["m_mir"], sc.info["m_mir"]]          # "the three efficiencies"
    # call 1: 293 blocks with a ragged tail; call 2: fewer photons, other ids, other factors -- it reuses the front of
    # the scratch and finds call 1's leftovers behind it
    calls = [dict(lo=0, n=600_000 - 37, seed=9, base=123_456_789, fac=fac),
             dict(lo=250_000, n=2048 * 11 + 5, seed=4, base=1 << 40, fac=fac[:2])]
    for c in calls:
        o, d, lam = w.photon_range(c["lo"], c["lo"] + c["n"])
        do, dd, dl = (torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (o, d, lam))
        ref = gs.prefilter(do, dd, dl, c["fac"], seed=c["seed"], photon_id_base=c["base"])      # existing path, own workspace
        got = gs.prefilter_noalloc(do, dd, dl, c["fac"], _caller_buffers(c["n"], 3.0), seed=c["seed"], photon_id_base=c["base"])
        torch.cuda.synchronize()
        k = int(ref["n_kept"].item())
        assert 0.05 * c["n"] < k < 0.5 * c["n"]
        assert int(got["n_kept"].item()) == k
        a, b = _bytes(got, k), _bytes(ref, k)
        for key in KEYS:
            assert np.array_equal(a[key], b[key]), key
        # nothing beyond the survivors was written
        assert bool((got["index"][k:] == -7).all()) and bool((got["wavelengths"][k:] == 3.0).all())


def test_the_limit_is_accepted_and_one_photon_more_is_refused_with_the_limit_in_the_message():
    sc = wl.make_config("C2", n=1).scene
    gs = pkg.Scene(sc).build()
    n = opx.PREFILTER_NOALLOC_MAX_PHOTONS + 1
    lam = torch.empty(n, dtype=torch.float32, device="cuda")       # only its length and address reach the call
    x3 = torch.empty((4, 3), dtype=torch.float32, device="cuda")
    out = _caller_buffers(4, 5.0)
    with pytest.raises(pkg.OpxError) as e:
        gs.prefilter_noalloc(x3, x3, lam, [sc.info["m_det"]], out)
    assert e.value.status == opx.OPX_ERR_INVALID_ARG and str(opx.PREFILTER_NOALLOC_MAX_PHOTONS) in str(e.value)
    torch.cuda.synchronize()
    assert int(out["n_kept"].item()) == 12345 and bool((out["wavelengths"] == 5.0).all())
    # the limit itself is accepted and fills the scratch array to its last block: same survivors as the workspace path
    n = opx.PREFILTER_NOALLOC_MAX_PHOTONS
    g = torch.Generator(device="cuda").manual_seed(5)
    o = torch.rand((n, 3), generator=g, device="cuda")
    d = torch.rand((n, 3), generator=g, device="cuda")
    lam = 200.0 + 400.0 * torch.rand(n, generator=g, device="cuda")
    fac = [sc.info["m_det"], sc.info["m_mir"]]
    cap = n // 2
    ref = gs.prefilter(o, d, lam, fac, seed=2, capacity=cap)
    got = gs.prefilter_noalloc(o, d, lam, fac, _caller_buffers(cap, 3.0), seed=2)
    torch.cuda.synchronize()
    k = int(ref["n_kept"].item())
    assert 0 < k < cap and int(got["n_kept"].item()) == k
    for key in KEYS:
        assert torch.equal(got[key][:k], ref[key][:k]), key
