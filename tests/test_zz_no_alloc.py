"""dm_probe_update_noalloc: the probe update (eq. (5)) for callers that cannot allocate.

Everything else in include/dm.h works out of a workspace the caller allocates and lends.  A caller that is not
allowed to allocate device memory (its host application gave the whole card to its own pool at start-up; or it
runs during a measurement, where the device-wide stall of cudaMalloc / cudaFree is not acceptable) has no
workspace, only the arrays it already owns.  For it the library carries a fixed 16 MiB array of its own for the
partial sums of the reduction (DM_NOALLOC_SCRATCH_BYTES; every GPU that loads the library holds it until exit).

What is checked here: the entry point returns the same probe as the probe step of dm_iterate (the existing,
workspace-backed path) within the one-step tolerance of the parity tests, on calls made one after the other
with DIFFERENT problem shapes -- the array is shared and keeps the previous call's contents, so a call that
relied on stale or zeroed contents would show up on the second or third call -- and problems beyond the fixed
size are refused with a text that says so.

The file is named to be collected last: `pytest -x` stops at the first failure, so a failure here cannot hide
another test.  It does not depend on what ran before it (fresh process or after the whole suite).
"""
import ctypes as C

import numpy as np
import pytest

from paper_1808_10375_b200 import build as dm_build
from paper_1808_10375_b200 import synth

TOL = 1e-5             # relative L2, the one-step bar of tests/test_gpu_parity.py
MAXABS_FACTOR = 10.0   # and max |delta| <= 10 TOL max |ref|, as there


@pytest.fixture(scope="module")
def dm():
    dm_build.build()
    from paper_1808_10375_b200 import dm as _dm
    _dm.lib()          # raises if the CUDA library is missing: there is no fallback
    return _dm


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _existing_path(dm, pr):
    """One dm_iterate on a workspace-backed plan; returns what its probe step read and what it wrote."""
    c = pr.cfg
    g = dm.DMPlan(c.N, c.n_views, c.K, c.L, c.obj_h, c.obj_w, pr.positions).alloc_workspace()
    g.set_data(_t(pr.intensities), _t(pr.probe0), _t(pr.object0))
    g.iterate(1)
    # the probe step of an iteration uses the NEW object and the NEW psi, and P_old = the probe before it
    got = dict(pos=_t(pr.positions.astype(np.int32)), O=g.object(), psi=g.psi(), P_old=_t(pr.probe0.astype(np.complex64)),
               alpha=g.alphas[1], P_new=g.probe(), chunks=g.geometry()["prb_chunks"])
    g.close()
    return got


def _check(dm, ref, out):
    import torch
    out.fill_(float("nan"))      # every element must be written by the call
    ret = dm.probe_update_noalloc(ref["pos"], ref["O"], ref["psi"], ref["P_old"], ref["alpha"], out=out)
    assert ret is out
    torch.cuda.synchronize()
    a, b = out.cpu().numpy().astype(np.complex128), ref["P_new"].cpu().numpy().astype(np.complex128)
    assert np.isfinite(a).all()
    r = synth.rel_l2(a, b)
    m = float(np.abs(a - b).max() / np.abs(b).max())
    assert r <= TOL and m <= MAXABS_FACTOR * TOL, (r, m)
    return out.cpu().numpy().copy(), r


@pytest.mark.gpu
def test_noalloc_probe_update_matches_plan_path_on_calls_in_a_row(dm):
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    # three shapes that lay the shared array out differently: (N, K, L) = (128, 2, 1), (256, 4, 2), (128, 4, 1);
    # the last has 100 views, where the fixed array holds fewer view chunks than the plan's workspace would
    problems = [synth.make_problem(synth.CONFIGS[1].scaled(6, 5)),
                synth.make_problem(synth.CONFIGS[3].scaled(3, 3)),
                synth.make_problem(synth.CONFIGS[2].scaled(10, 10))]
    refs = [_existing_path(dm, pr) for pr in problems]
    outs = [torch.empty_like(r["P_new"]) for r in refs]
    c2 = problems[2].cfg
    per_chunk = c2.N * c2.N * (8 * c2.K + 4)
    assert refs[2]["chunks"] > dm.NOALLOC_SCRATCH_BYTES // per_chunk, "case 3 is meant to be limited by the fixed array"
    first = []
    for ref, out in zip(refs, outs):                  # calls in a row, no clearing in between
        first.append(_check(dm, ref, out)[0])
    for ref, out, f in zip(refs, outs, first):        # and again, now over the last call's leftovers
        again, _ = _check(dm, ref, out)
        assert np.array_equal(again, f), "the result depends on what an earlier call left in the shared array"


@pytest.mark.gpu
def test_noalloc_literal_quotient_and_uncovered_probe(dm):
    """alpha = 0 (the literal quotient of eq. (5)) with an all-zero object: every denominator is 0, so the probe
    must come back unchanged -- right after a call that left non-zero partial sums in the array."""
    import torch
    pr = synth.make_problem(synth.CONFIGS[1].scaled(3, 3))
    ref = _existing_path(dm, pr)
    out = torch.empty_like(ref["P_new"])
    _check(dm, ref, out)
    zero_O = torch.zeros_like(ref["O"])
    dm.probe_update_noalloc(ref["pos"], zero_O, ref["psi"], ref["P_old"], 0.0, out=out)
    torch.cuda.synchronize()
    assert torch.equal(out, ref["P_old"])


def test_noalloc_refuses_what_does_not_fit(dm):
    """Argument and size checks come before the first CUDA call, so they run without a GPU: a problem whose
    partial sums exceed the fixed array is refused with DM_ERR_WORKSPACE and a text naming both sizes."""
    L = dm.lib()
    dummy = C.c_void_p(256)            # never dereferenced: the call is refused first
    err = C.create_string_buffer(512)

    def call(N, n_views, K, Lm, H, W, alpha=0.0, ptr=dummy):
        return L.dm_probe_update_noalloc(N, n_views, K, Lm, H, W, ptr, ptr, ptr, ptr, alpha, ptr, None, err, len(err))

    assert 512 * 512 * (8 * 8 + 4) > dm.NOALLOC_SCRATCH_BYTES
    assert call(512, 10, 8, 1, 600, 600) == 5
    text = err.value.decode()
    assert str(512 * 512 * (8 * 8 + 4)) in text and str(dm.NOALLOC_SCRATCH_BYTES) in text, text
    assert call(96, 10, 1, 1, 600, 600) == 3 and "N = 96" in err.value.decode()
    assert call(64, 10, 3, 3, 600, 600) == 3
    assert call(64, 0, 1, 1, 600, 600) == 1
    assert call(64, 10, 1, 1, 600, 600, alpha=-1.0) == 1
    assert call(64, 10, 1, 1, 32, 600) == 2
    assert call(64, 10, 1, 1, 600, 600, ptr=None) == 1
    # and a NULL text buffer is allowed
    assert L.dm_probe_update_noalloc(96, 1, 1, 1, 600, 600, dummy, dummy, dummy, dummy, 0.0, dummy, None, None, 0) == 3
