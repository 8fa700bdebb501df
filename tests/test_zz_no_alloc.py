"""psc_marder_static against psc_marder (include/psc.h).

psc_marder_static exists for users who may not allocate device memory at the point where they
apply Marder's correction: a time loop running while another thread captures a CUDA graph in the
global mode (cudaMalloc is forbidden there), a loop that cannot take cudaMalloc's device-wide
synchronisation, a process whose own pool already owns the HBM.  Its rho / residual scratch is a
fixed array inside the library (PSC_MARDER_STATIC_MAX_POINTS grid points incl. ghosts) that every
call on the device shares and that keeps the previous call's contents -- which is exactly what can
go wrong and what these tests look at: the second of two calls in a row, a small grid right after
a large one, the size limit, and that the device's free memory does not move.

The file name sorts after every other test file on purpose: pytest -x stops at the first failure,
and a failure here must not hide the parity tests.  Nothing here depends on what ran before it in
the process (the array's contents are never assumed), so it passes alone and at the end of the
whole suite.
"""
import numpy as np
import pytest
import torch

import paper_1310_7866_b200 as psc
import psc_inputs
from tests.util import rel_maxnorm, smooth_fields

pytestmark = pytest.mark.gpu
TOL = 1e-5      # the tolerance of tests/test_gpu_marder.py: max-norm per component of E


def _sim(pl, **kw):
    from paper_1310_7866_b200.harness import Simulation

    return Simulation(pl, **kw)


def _plasma(kind):
    if kind == "2d":
        pl = psc_inputs.make_config(1)
    elif kind == "3d":
        pl = psc_inputs.thermal((12, 20, 8), 5, seed=12, dx=(0.8, 1.25, 0.5), name="3d")
    else:                                   # order 2, 3-d
        pl = psc_inputs.make_config(5, scale=(8, 8, 32))
    return smooth_fields(pl, 0.05, seed=33)  # E not consistent with rho: a large Gauss residual


def _diffusion(pl, frac=0.8):
    return frac / sum(4.0 / pl.dx[d] ** 2 for d in range(3) if pl.n[d] > 1)


def _interior(sim):
    return sim.interior(sim.E).cpu().numpy()


def _pair(kind):
    """two contexts on the same seeded state: `a` takes psc_marder, `b` psc_marder_static"""
    a, b = _sim(_plasma(kind)), _sim(_plasma(kind))
    a.psc.particles_sort()
    b.psc.particles_sort()
    assert torch.equal(a.E, b.E)
    return a, b


@pytest.mark.parametrize("kind", ["2d", "3d", "beam"])
def test_marder_static_matches_marder_on_two_calls_in_a_row(kind):
    """call 1 and, straight after it, call 2 (which finds call 1's rho and residual still in the
    array); then two time steps -- some particles now wait in exchange rows, rho has changed -- and
    a third call.  After every call E of the static path agrees with E of psc_marder within the
    Marder tests' tolerance; the correction really changes E each time; ghosts stay periodic images."""
    a, b = _pair(kind)
    D = _diffusion(a.plasma)
    E_prev = _interior(b)
    for call, iters in enumerate((3, 2)):
        a.psc.marder(D, iters)
        b.psc.marder_static(D, iters)
        Ea, Eb = _interior(a), _interior(b)
        assert rel_maxnorm(Eb, Ea.astype(np.float64)) < TOL, (kind, call)
        assert np.abs(Eb - E_prev).max() > 10 * TOL * np.abs(Eb).max(), (kind, call)   # not a no-op
        E_prev = Eb
    a.step(2)
    b.step(2)
    a.psc.marder(D, 1)
    b.psc.marder_static(D, 1)
    assert rel_maxnorm(_interior(b), _interior(a).astype(np.float64)) < TOL, kind
    G = b.E.clone()
    b.psc.fill_ghosts(psc.PSC_E)
    assert torch.equal(G, b.E)
    assert a.psc.status() == 0 and b.psc.status() == 0


def test_marder_static_small_grid_after_a_large_one():
    """the array is shared by all contexts of the device: a 3-d context fills it, then a much
    smaller 2-d context (other extents, other strides) uses it, twice, then the 3-d one again"""
    big_a, big_b = _pair("beam")
    small_a, small_b = _pair("2d")
    Db, Ds = _diffusion(big_a.plasma), _diffusion(small_a.plasma)
    for _ in range(2):
        big_a.psc.marder(Db, 2)
        big_b.psc.marder_static(Db, 2)
        for _ in range(2):
            small_a.psc.marder(Ds, 2)
            small_b.psc.marder_static(Ds, 2)
            assert rel_maxnorm(_interior(small_b), _interior(small_a).astype(np.float64)) < TOL
        assert rel_maxnorm(_interior(big_b), _interior(big_a).astype(np.float64)) < TOL


def test_marder_static_size_limit_and_the_largest_grid_that_fits():
    """ex*ey*ez <= PSC_MARDER_STATIC_MAX_POINTS is served (1 x 568 x 568 cells: 572^2 = 327 184 points
    of 327 680), one more row of blocks is refused with PSC_ERR_SCRATCH_LIMIT and E is not touched;
    the argument checks it shares with psc_marder come first and give the same codes"""
    fits = psc_inputs.thermal((1, 568, 568), 1, seed=5, name="fits")
    smooth_fields(fits, 0.05, seed=34)
    a, b = _sim(fits), _sim(fits)
    assert a.psc.ext[0] * a.psc.ext[1] * a.psc.ext[2] <= psc.MARDER_STATIC_MAX_POINTS
    D = _diffusion(fits)
    L = psc.lib()
    assert L.psc_marder_static(b.psc._h, None, D, 1) == -3          # PSC_ERR_NOT_SORTED, as psc_marder
    assert L.psc_marder(a.psc._h, None, D, 1) == -3
    a.psc.particles_sort()
    b.psc.particles_sort()
    assert L.psc_marder_static(b.psc._h, None, 1.3 * D / 0.8, 1) == -4   # PSC_ERR_CFL
    assert L.psc_marder_static(b.psc._h, None, D, -1) == -1              # PSC_ERR_INVALID_ARG
    for _ in range(2):
        a.psc.marder(D, 2)
        b.psc.marder_static(D, 2)
        assert rel_maxnorm(_interior(b), _interior(a).astype(np.float64)) < TOL
    del a, b

    over = psc_inputs.thermal((1, 576, 576), 1, seed=6, name="over")   # 580^2 = 336 400 points
    smooth_fields(over, 0.05, seed=35)
    c = _sim(over)
    assert c.psc.ext[0] * c.psc.ext[1] * c.psc.ext[2] > psc.MARDER_STATIC_MAX_POINTS
    c.psc.particles_sort()
    E0 = c.E.clone()
    assert L.psc_marder_static(c.psc._h, None, _diffusion(over), 1) == psc.PSC_ERR_SCRATCH_LIMIT
    assert b"psc_marder_static" in L.psc_strerror(psc.PSC_ERR_SCRATCH_LIMIT)
    torch.cuda.synchronize()
    assert torch.equal(E0, c.E)
    with pytest.raises(psc.PscError):
        c.psc.marder_static(_diffusion(over), 1)
    c.psc.marder(_diffusion(over), 1)        # the allocating call has no such limit
    torch.cuda.synchronize()
    assert not torch.equal(E0, c.E)


def test_marder_static_leaves_the_free_device_memory_alone():
    """cudaMemGetInfo before and after: psc_marder's first call takes its scratch field from the
    device, psc_marder_static's calls take nothing (the first call of each, which also loads the
    kernels, is done before the measurement)"""
    pl = psc_inputs.thermal((64, 64, 64), 1, seed=9, name="mem")      # scratch field: 3 * 68^3 floats = 3.8 MB
    smooth_fields(pl, 0.05, seed=36)
    a, b = _sim(pl), _sim(pl)
    a.psc.particles_sort()
    b.psc.particles_sort()
    D = _diffusion(pl)
    b.psc.marder_static(D, 1)             # set-up call: symbol address, module / kernel loading
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        b.psc.marder_static(D, 2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    a.psc.marder(D, 1)                    # for contrast: this one allocates (outside torch's pool)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] < free0
