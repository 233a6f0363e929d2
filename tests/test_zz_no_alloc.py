"""chim_build_pcat_static: p_cat from galaxy lists (eq. 8) for callers that must not allocate on the GPU.

Who needs it: a sampler that shares its process with JAX or PyTorch, where the framework's pool already holds nearly all of
the device memory (a cudaMalloc from libchim then fails), and a loop that rebuilds p_cat between likelihood batches, where
the device-wide synchronisation of cudaMalloc / cudaFree would stall the batch still in flight.  The entry point takes device
pointers for everything and keeps its per-galaxy scratch in a fixed 2 MiB array inside libchim.so
(CHIM_PCAT_STATIC_MAX_GALAXIES galaxies per call), which all calls on a GPU share.

What is checked here: its output equals that of the existing allocating path, chim_build_pcat, at the tolerance the p_cat
parity tests use (rtol 1e-10), on two calls in a row with different inputs -- the second call finds the first call's
coefficients still in the array and must not be affected by them -- and a call beyond the limit is refused with a message.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity tests.
It passes alone in a fresh process (the first call does the array's address look-up) and after the other GPU tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

RTOL = 1e-10          # as test_build_pcat_matches_the_oracle_and_feeds_the_path
ATOL = 1e-290


@pytest.fixture(scope="module")
def P():
    import paper_2504_02034_b200 as pkg
    pkg.lib()                      # fails loudly if libchim.so is missing
    return pkg


def _catalogue(seed, ngal, nz, z_lo):
    """Galaxy lists and grids per line of sight: spectroscopic and photometric widths mixed, ragged sizes."""
    rng = np.random.default_rng(seed)
    gal_off = np.concatenate([[0], np.cumsum(ngal)]).astype(np.int64)
    z_gal = np.concatenate([rng.uniform(0.05, 1.4, n) for n in ngal])
    sig = np.where(rng.random(z_gal.size) < 0.5, 0.001, 0.03) * (1 + z_gal)
    wg = rng.uniform(0.3, 3.0, z_gal.size)
    grid_off = np.concatenate([[0], np.cumsum(nz)]).astype(np.int64)
    z_grid = np.concatenate([np.linspace(lo, lo + 0.9, n) for lo, n in zip(z_lo, nz)])
    return gal_off, z_gal, sig, wg, grid_off, z_grid


def _static(c, torch, om, gal_off, z_gal, sig, wg, grid_off, z_grid):
    dev = c.device
    d = lambda a: torch.as_tensor(a, device=dev).contiguous()        # the caller's own device buffers (torch's allocator)
    out = torch.full((z_grid.size,), -1.0, dtype=torch.float64, device=dev)
    c.build_pcat_static(om, int(gal_off[-1]), d(gal_off), d(z_gal), d(sig), d(grid_off), d(z_grid), out,
                        w_gal=None if wg is None else d(wg))
    torch.cuda.synchronize()
    return out.cpu().numpy()


def test_static_scratch_entry_point_matches_the_allocating_path_on_two_calls_in_a_row(P):
    import torch
    c = P.Context()
    # call 1: five lines of sight, weighted; call 2: other sizes, another Omega_m, unit weights, MORE galaxies per line of
    # sight at the start of the array and fewer overall -- so stale coefficients of call 1 sit both under and beyond call 2's
    first = _catalogue(17, [1, 50, 500, 333, 7], [300, 1000, 257, 4096, 2], (0.0, 0.1, 0.3, 0.2, 0.5))
    second = _catalogue(23, [64, 3, 290], [513, 31, 1200], (0.2, 0.0, 0.4))
    worst = 0.0
    for om, (gal_off, z_gal, sig, wg, grid_off, z_grid), w_in in ((0.31, first, True), (0.27, second, False)):
        wg_in = wg if w_in else None
        got = _static(c, torch, om, gal_off, z_gal, sig, wg_in, grid_off, z_grid)
        ref = c.build_pcat(om, gal_off, z_gal, sig, grid_off, z_grid, w_gal=wg_in)       # the existing path (allocates, validates)
        assert np.all(np.isfinite(got)) and got.shape == ref.shape
        assert np.allclose(got, ref, rtol=RTOL, atol=ATOL)
        nz = ref > 1e-280
        worst = max(worst, float(np.max(np.abs(got[nz] - ref[nz]) / ref[nz])))
    assert worst < RTOL
    # the first call again after the second one: same answer as before, whatever the array held in between
    gal_off, z_gal, sig, wg, grid_off, z_grid = first
    again = _static(c, torch, 0.31, gal_off, z_gal, sig, wg, grid_off, z_grid)
    assert np.allclose(again, c.build_pcat(0.31, gal_off, z_gal, sig, grid_off, z_grid, w_gal=wg), rtol=RTOL, atol=ATOL)
    c.close()


def test_static_scratch_entry_point_refuses_what_the_array_cannot_hold(P):
    import torch
    c = P.Context()
    gal_off, z_gal, sig, wg, grid_off, z_grid = _catalogue(5, [10, 20], [40, 50], (0.1, 0.2))
    dev = c.device
    d = lambda a: torch.as_tensor(a, device=dev).contiguous()
    out = torch.zeros(z_grid.size, dtype=torch.float64, device=dev)
    with pytest.raises(P.ChimError) as ei:          # the size the caller states is beyond the fixed array: refused before any launch
        c.build_pcat_static(0.3, P.CHIM_PCAT_STATIC_MAX_GALAXIES + 1, d(gal_off), d(z_gal), d(sig), d(grid_off), d(z_grid), out)
    assert "CHIM_PCAT_STATIC_MAX_GALAXIES" in str(ei.value) and str(P.CHIM_PCAT_STATIC_MAX_GALAXIES) in str(ei.value)
    with pytest.raises(P.ChimError):
        c.build_pcat_static(1.5, int(gal_off[-1]), d(gal_off), d(z_gal), d(sig), d(grid_off), d(z_grid), out)      # Omega_m > 1
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0            # nothing ran
    # offsets that disagree with the stated total: that line of sight comes back NaN, the array is not left, the other is right
    c.build_pcat_static(0.3, 10, d(gal_off), d(z_gal), d(sig), d(grid_off), d(z_grid), out)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    ref = c.build_pcat(0.3, gal_off, z_gal, sig, grid_off, z_grid)
    assert np.allclose(got[:40], ref[:40], rtol=RTOL, atol=ATOL) and np.all(np.isnan(got[40:]))
    c.close()
