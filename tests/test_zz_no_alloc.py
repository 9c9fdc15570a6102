"""gray_shadow_edge_noalloc: the shadow statistics for a caller that may not allocate device memory.

Some users of libgray run on a GPU whose memory is not theirs to manage: a plug-in that a host program hands its
buffers to and forbids cudaMalloc (the host's own pool holds the whole device), a worker whose fixed memory slice is
already filled by the photon buffers, a frame loop that cannot stall on cudaMalloc / cudaFree.  They have no
workspace to give gray_shadow_edge, so gray_shadow_edge_noalloc keeps its scratch memory in an array built into
libgray.so (128.5 KB per GPU, at most GRAY_NOALLOC_MAX_ANGLES = 16384 spokes; include/gray.h).

What is checked: on two calls in a row, with different images and spoke counts so that the second call finds the
first one's leftovers in the shared array, the entry point returns what gray_shadow_edge returns on the same batch,
at the tolerance the shadow tests of test_gpu_parity.py use (1e-12; the captured count exactly); a spoke count over
the limit is refused by name; and the workspace of the batch is never touched.

This file is collected last on purpose (`pytest --collect-only`): under `pytest -x` a failure here hides nothing.
It needs no state from the other tests and leaves none: it passes alone in a fresh process (where its first call is
the one that looks the array's address up) and after the whole suite.
"""
import ctypes

import pytest
import torch

import paper_1303_5057_b200 as g
from paper_1303_5057_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-12          # tests/test_gpu_parity.py::test_classify_and_shadow_edge_match_oracle_and_bardeen
KEYS = ("area", "centroid_alpha", "centroid_beta", "alpha_min", "alpha_max", "D", "R_mean", "A")


def _image(a, inc, W, nx, ny):
    b = g.PhotonBatch(nx * ny)
    g.gray_init_rays(b, a, wl.R_OBS, inc, W, nx, ny)
    g.gray_integrate(b, params=g.StepParams(rule=g.STEP_EQ2))
    return b


def _same(b, n_angles):
    """The no-alloc entry point against the existing path on one batch; returns the no-alloc result."""
    r_ref = torch.full((max(n_angles, 1),), -1.0, dtype=torch.float64, device="cuda")
    r_new = torch.full((max(n_angles, 1),), -2.0, dtype=torch.float64, device="cuda")
    ref = g.gray_shadow_edge(b, n_angles, r_ref)
    b.workspace.fill_(0xA5)                       # the no-alloc call must neither need nor touch the workspace
    new = g.gray_shadow_edge_noalloc(b, n_angles, r_new)
    assert bool((b.workspace == 0xA5).all())
    assert new["n_captured"] == ref["n_captured"]
    for k in KEYS:
        assert abs(new[k] - ref[k]) <= TOL * max(1.0, abs(ref[k])), (k, new[k], ref[k])
    if n_angles:
        assert float((r_new[:n_angles] - r_ref[:n_angles]).abs().max()) <= TOL
    assert g.gray_shadow_edge_noalloc(b, n_angles)["R_mean"] == new["R_mean"]      # radius_dev is optional
    return new


def test_two_calls_in_a_row_match_the_workspace_path():
    # first call: a wide Kerr shadow, more spokes than gray_shadow_edge keeps in shared memory (5120), a ragged grid
    big = _image(0.9, 60.0, 10.0, 160, 131)
    first = _same(big, 6000)
    assert first["n_captured"] > 1000
    # second call right after it: a smaller Schwarzschild shadow in a wider field, fewer spokes.  Every sum, the
    # captured count, the extreme columns and the radii of the first call are still in the array when it starts.
    small = _image(0.0, 30.0, 14.0, 96, 96)
    second = _same(small, 360)
    assert 0 < second["n_captured"] < first["n_captured"]
    assert second["alpha_max"] - second["alpha_min"] > 9.0      # 2 sqrt(27) = 10.39 less two pixels of 0.29
    # and the first image once more: the result does not depend on what ran in between
    again = g.gray_shadow_edge_noalloc(big, 6000)
    assert again == first


def test_limit_and_argument_errors_are_reported_before_any_launch():
    limit = g.gray_noalloc_max_angles()
    assert limit == 16384
    b = g.PhotonBatch(20 * 15)
    g.gray_init_rays(b, 0.5, wl.R_OBS, 60.0, 10.0, 20, 15)
    b.status.fill_(g.ESCAPED)
    b.status[7 * 20 + 9] = g.CAPTURED                                   # one captured pixel
    at_limit = g.gray_shadow_edge_noalloc(b, limit)                     # the largest size is accepted ...
    assert at_limit["n_captured"] == 1
    ref = g.gray_shadow_edge(b, limit)
    for k in KEYS:
        assert abs(at_limit[k] - ref[k]) <= TOL * max(1.0, abs(ref[k])), k
    with pytest.raises(g.GrayError, match="GRAY_NOALLOC_MAX_ANGLES"):    # ... one more is refused, by name
        g.gray_shadow_edge_noalloc(b, limit + 1)
    s = g.gray._ShadowStats()
    rc = g.lib().gray_shadow_edge_noalloc(ctypes.byref(b.c), limit + 1, None, ctypes.byref(s), None)
    assert rc == -1 and b"16384" in g.lib().gray_last_error()
    empty = g.gray_shadow_edge_noalloc(b, 0)                             # no spokes: area and centroid only
    assert empty["n_captured"] == 1 and empty["R_mean"] == 0.0 and empty["A"] == 0.0
    br = g.PhotonBatch(64)
    g.gray_init_rays_random(br, 0.5, wl.R_OBS, 60.0, 10.0, 1)
    with pytest.raises(g.GrayError):
        g.gray_shadow_edge_noalloc(br, 16)                               # random pixels have no image grid
