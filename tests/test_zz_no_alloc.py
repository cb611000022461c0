"""adept_raycast_batch_static (include/adept.h): the ray-cast validator with its device buffers in the library's
file-scope scratch array instead of cudaMalloc'ed memory.  Same kernel, so the results must equal
adept_raycast_batch's -- on two calls in a row, because the array keeps what the last call left in it.

Collected last on purpose (the name): a failure here must not hide the parity tests from `pytest -x`.  Runs alone
in a fresh process and after the other tests alike: it needs nothing but its own context."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _patch_rays(rng, n):
    """Rays from the origin into and around the 12 x 12 crystal patch; the last few start outside the world."""
    phi = rng.uniform(-0.05, 0.26, n)
    eta = rng.uniform(-0.15, 0.15, n)
    th = 2.0 * np.arctan(np.exp(-eta))
    d = np.stack([np.sin(th) * np.cos(phi), np.sin(th) * np.sin(phi), np.cos(th)], axis=1)
    pos = np.zeros_like(d)
    pos[-3:] = [400.0, 0.0, 0.0]
    return pos, d


def _same(static, plain):
    col_s, nx_s = static
    col, nx = plain[0], plain[1]
    assert np.array_equal(nx_s, nx)                                   # boundaries crossed: exact
    np.testing.assert_allclose(col_s, col, rtol=1e-12, atol=1e-12)    # the ray-cast tests' tolerance (test_gpu_navigation.py)


def test_static_scratch_raycast_equals_the_allocating_one_on_calls_in_a_row(barrel_patch):
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field
    g, _, tabs, scal = barrel_patch
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10)
    rng = np.random.default_rng(2209)
    # first call: several tiles and a ragged tail; second call: fewer, different rays (what the first left behind in
    # the array lies beyond them and under them); third: the single-precision geometry, fewer crossings allowed
    p1, d1 = _patch_rays(rng, 4099)
    p2, d2 = _patch_rays(rng, 777)
    r1 = a.raycast_static(p1, d1, adept.NAV_BVH)
    r2 = a.raycast_static(p2, d2, adept.NAV_BVH)
    _same(r1, a.raycast(p1, d1, adept.NAV_BVH))
    _same(r2, a.raycast(p2, d2, adept.NAV_BVH))
    assert r1[1][:-3].max() >= 8 and (r1[1][-3:] == -1).all() and (r2[1][-3:] == -1).all()
    assert not np.array_equal(r1[0][:777], r2[0])
    # the same two batches again, in the other order, with the loop navigator and a stream of the caller's
    import torch
    st = torch.cuda.Stream(device=a.device)
    r2b = a.raycast_static(p2, d2, adept.NAV_LOOP, stream=st)
    r1b = a.raycast_static(p1, d1, adept.NAV_LOOP, stream=st)
    _same(r2b, r2)
    _same(r1b, r1)
    r3 = a.raycast_static(p2, d2, adept.NAV_BVH_F32, max_crossings=5)
    _same(r3, a.raycast(p2, d2, adept.NAV_BVH_F32, max_crossings=5))
    assert r3[1].max() == 5
    a.close()


def test_static_scratch_limits(barrel_patch):
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field
    g, _, tabs, scal = barrel_patch
    a = adept.Adept(g, tabs, scal, field.no_field(), track_capacity=1 << 10)
    rng = np.random.default_rng(15445)
    n = adept.STATIC_MAX_RAYS
    p, d = _patch_rays(rng, n + 1)
    with pytest.raises(adept.AdeptError) as err:                      # one ray too many: refused, nothing launched
        a.raycast_static(p, d)
    assert "ADEPT_STATIC_MAX_RAYS" in str(err.value) and str(n) in str(err.value)
    col, nx = a.raycast_static(p[:0], d[:0])                          # no rays: nothing to do
    assert col.shape == (0,) and nx.shape == (0,)
    full = a.raycast_static(p[:n], d[:n])                             # the whole array in use
    _same(full, a.raycast(p[:n], d[:n]))
    one = a.raycast_static(p[5:6], d[5:6])                            # ... and one ray after it
    assert one[1][0] == full[1][5] and one[0][0] == full[0][5]
    a.close()
