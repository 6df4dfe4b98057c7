"""GPU test of mhd_max_divb_noalloc (csrc/mhd_noalloc.cu): the div B diagnostic with its reduction scratch
in a static __device__ array, for callers that may not allocate.  Checked against the existing path
(mhd_max_divb on a context holding the same state) and against the definition in numpy, on calls in a row
that share the scratch array: a large grid first, then a small one whose maximum is smaller (stale partial
maxima of the first call must not be read), then the large one again.  Named test_zz_* so that pytest
collects it last."""
import numpy as np
import pytest

from paper_2402_05240_b200 import inputs
from helpers import FIELDS

pytestmark = pytest.mark.gpu
TOL_DIVB = 1e-12   # the tolerance of the div B checks in tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def mhd():
    from paper_2402_05240_b200 import mhd as m
    return m


def make_state(n, seed, amplitude, periodic):
    """A physical state whose face field is NOT solenoidal (random faces), so that max |div B| is a number
    of order amplitude * n and not round-off."""
    p = inputs.random_smooth(n=n, seed=seed, recon=1)
    rng = np.random.default_rng(seed)
    st = {f: np.ascontiguousarray(p.state[f]) for f in FIELDS}
    for f in ("bx", "by", "bz"):
        st[f] = amplitude * rng.standard_normal(st[f].shape)
    if periodic:   # face n is face 0 on a periodic axis (mhd_set_state keeps only faces 0 .. n-1)
        st["bx"][:, :, -1] = st["bx"][:, :, 0]; st["by"][:, -1, :] = st["by"][:, 0, :]; st["bz"][-1, :, :] = st["bz"][0, :, :]
    return p.gamma, st


def divb_numpy(st, n):
    d = [1.0 / n[a] for a in range(3)]
    div = ((st["bx"][:, :, 1:] - st["bx"][:, :, :-1]) / d[0] + (st["by"][:, 1:, :] - st["by"][:, :-1, :]) / d[1]
           + (st["bz"][1:, :, :] - st["bz"][:-1, :, :]) / d[2])
    return float(np.abs(div).max())


def existing_path(mhd, n, gamma, st, bc):
    g = mhd.Mhd(*n, gamma, 1, bc)
    g.set_state(st)
    v = g.max_divb()
    g.close()
    return v


def test_no_alloc_divb_matches_the_existing_path_on_calls_in_a_row(mhd):
    import torch
    dev = torch.device("cuda:0")
    cases = [((96, 64, 40), 5, 1.0, True), ((9, 7, 5), 6, 1e-3, False), ((96, 64, 40), 7, 0.5, False)]
    prepared = []
    for n, seed, amp, periodic in cases:
        gamma, st = make_state(n, seed, amp, periodic)
        want = existing_path(mhd, n, gamma, st, (0, 0, 0) if periodic else (1, 1, 1))
        assert abs(want - divb_numpy(st, n)) <= TOL_DIVB * want      # the existing path is the definition
        prepared.append((n, st, want, {f: torch.from_numpy(st[f]).to(dev) for f in ("bx", "by", "bz")}))
    assert prepared[1][2] < 1e-2 * prepared[0][2]                     # the second maximum lies far below the first
    out = torch.full((len(cases),), -1.0, dtype=torch.float64, device=dev)
    stream = torch.cuda.Stream()
    torch.cuda.synchronize()
    mem0 = torch.cuda.memory_allocated()
    for q, (n, st, want, t) in enumerate(prepared):                   # back to back on one stream, no sync between
        mhd.max_divb_noalloc(n, [1.0 / n[a] for a in range(3)], t["bx"], t["by"], t["bz"], out[q:q + 1], stream)
    stream.synchronize()
    assert torch.cuda.memory_allocated() == mem0
    got = out.cpu().numpy()
    for q, (n, st, want, t) in enumerate(prepared):
        assert abs(got[q] - want) <= TOL_DIVB * want, (q, n, got[q], want)


def test_no_alloc_divb_rejects_grids_beyond_the_static_scratch(mhd):
    import torch
    dev = torch.device("cuda:0")
    t = torch.zeros(8, dtype=torch.float64, device=dev)
    out = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
    assert 256 * 256 * 256 == mhd.NOALLOC_MAX_CELLS
    with pytest.raises(mhd.MhdError, match="exceed the static scratch"):
        mhd.max_divb_noalloc((257, 256, 256), (1.0, 1.0, 1.0), t, t, t, out)
    with pytest.raises(mhd.MhdError, match="bad grid size"):
        mhd.max_divb_noalloc((4, 0, 4), (1.0, 1.0, 1.0), t, t, t, out)
    torch.cuda.synchronize()
    assert float(out.cpu()[0]) == -1.0                                 # nothing was launched
