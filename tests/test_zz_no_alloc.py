"""GPU test of the allocation-free entry point jf_plane_sums_static (include/jf.h): jf_plane_sums with its partial sums
in a static device array inside the library instead of the solver's workspace, for callers that must not allocate.
Checked against the existing path (jf_plane_sums, itself checked against the numpy oracle in tests/test_gpu_stats.py) on
two calls in a row, at the tolerance of tests/test_gpu_stats.py (1e-12 in fp64, 1e-5 for fp32 states; the two paths run
the same kernels in the same order, so they in fact agree bit for bit).  Named test_zz_* so that pytest collects it last."""
import numpy as np
import pytest

from paper_2406_19494_b200 import cases

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-12, "f32": 1e-5}


@pytest.fixture(scope="module")
def jf():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2406_19494_b200 import binding
    binding.lib()
    return binding


def _close(a, b, tol):
    a, b = a.cpu().numpy(), b.cpu().numpy()
    scale = np.maximum(np.max(np.abs(b), axis=1, keepdims=True), 1e-300)
    return np.max(np.abs(a - b) / scale) <= tol


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_static_scratch_entry_point_matches_the_workspace_path_on_two_calls_in_a_row(jf, dtype):
    import torch
    c = cases.channel(48, 32, 24, n_steps=1)                  # stretched wall-normal axis: area weights matter
    s = jf.Solver(c, dtype)
    U = s.state()
    outs = [torch.empty((14, c.n[a]), dtype=torch.float64, device=s.device) for a in range(3)]
    # call 1: the axis with the MOST planes first, so that the shared array is left full of that call's partials ...
    for axis in (0, 1, 2):
        ref = s.jf_plane_sums(U, axis)
        got = s.jf_plane_sums_static(U, axis, outs[axis])
        assert _close(got, ref, TOL[dtype]), (dtype, axis, "first call")
        assert torch.equal(got, ref)                          # same kernels, same order: the same bits
    # ... call 2, directly after it, on another state and with fewer planes: stale contents must not leak into it
    s.jf_rk3_step(U, 1e-4)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for axis in (2, 1, 0):
        got = s.jf_plane_sums_static(U, axis, outs[axis])
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] >= free0          # the call took no device memory
        ref = s.jf_plane_sums(U, axis)
        assert _close(got, ref, TOL[dtype]), (dtype, axis, "second call")
        assert torch.equal(got, ref)
    # two solvers share the array: a call of one between two calls of the other (same stream) changes nothing
    c2 = cases.tgv(32)
    s2 = jf.Solver(c2, dtype)
    U2 = s2.state()
    a = s.jf_plane_sums_static(U, 1).clone()
    b2 = s2.jf_plane_sums_static(U2, 0)
    assert torch.equal(b2, s2.jf_plane_sums(U2, 0))
    assert torch.equal(s.jf_plane_sums_static(U, 1), a)


def test_static_scratch_entry_point_rejects_sizes_beyond_its_maximum(jf):
    L = jf.lib()
    nmax = L.jf_plane_sums_static_max_planes()
    assert nmax == 1024
    c = cases.random_admissible(n=(nmax + 4, 4, 4), seed=3)
    s = jf.Solver(c, "f64")
    U = s.state()
    with pytest.raises(jf.JFError) as e:
        s.jf_plane_sums_static(U, 0)                          # 1028 planes along x: beyond the static array
    assert e.value.status == jf.JF_EINVAL and "1024" in str(e.value) and "jf_plane_sums" in str(e.value)
    import torch
    assert torch.equal(s.jf_plane_sums_static(U, 1), s.jf_plane_sums(U, 1))   # 4 planes along y: fine
    assert s.jf_plane_sums(U, 0).shape == (14, nmax + 4)                       # the workspace path has no such limit
    c = cases.random_admissible(n=(nmax, 4, 4), seed=3)                        # exactly the maximum is accepted
    s = jf.Solver(c, "f64")
    U = s.state()
    assert torch.equal(s.jf_plane_sums_static(U, 0), s.jf_plane_sums(U, 0))
