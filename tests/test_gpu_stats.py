"""GPU parity of jf_plane_sums (plane statistics, PAPER.md:92-96 / Fig. 1) against the
numpy oracle oracle/stats.py on the same seeded inputs.  Floating-point sums in a different order: 1e-12 of the
plane's sum of |phi| dA in fp64; fp32 states against the same fp64 definition at 1e-5."""
import numpy as np
import pytest

from paper_2406_19494_b200 import cases

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def jf():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2406_19494_b200 import binding
    binding.lib()
    return binding


CASES = {
    "channel": lambda: cases.channel(48, 32, 32, n_steps=1),                       # stretched y, noise
    "ragged": lambda: cases.random_admissible(n=(70, 35, 67), seed=9, stretched=True),
    "tiny": lambda: cases.random_admissible(n=(4, 4, 4), seed=10),
    "tgv64": lambda: cases.tgv(64),
}


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_plane_sums_match_the_oracle(jf, name, axis, dtype):
    from oracle import stats
    c = CASES[name]()
    s = jf.Solver(c, dtype)
    U = s.state()
    got = s.jf_plane_sums(U, axis).cpu().numpy()
    again = s.jf_plane_sums(U, axis).cpu().numpy()
    assert np.array_equal(got, again)                                            # deterministic reduction
    Uh = U.cpu().numpy().astype(np.float64)                                      # the state the GPU saw (fp32 rounded)
    ref = stats.plane_sums(c, Uh, axis)
    assert got.shape == ref.shape == (14, c.n[axis])
    # scale of each sum: the same sum with |phi| (computed by the oracle on absolute values is not available
    # for products, so use the Cauchy-Schwarz-safe bound sqrt(S_{phi^2} S_1) >= |S_phi| via the quadratic rows)
    area = ref[0]
    scale = np.maximum(np.abs(ref), 1e-300)
    scale[3:6] = np.sqrt(ref[6:9] * area)                                        # u, v, w  <- uu, vv, ww
    scale[9] = np.sqrt(ref[6] * ref[7]); scale[10] = np.sqrt(ref[6] * ref[8]); scale[11] = np.sqrt(ref[7] * ref[8])
    scale = np.maximum(scale, 1e-300)                                           # identically-zero rows (w = 0 in the TGV)
    tol = 1e-12 if dtype == "f64" else 1e-5
    err = np.max(np.abs(got - ref) / scale)
    assert err <= tol, (name, axis, dtype, err)


def test_channel_profiles_from_device_sums(jf):
    """The Fig.-1 quantities of the seeded channel input: mean u follows the Poiseuille profile within the
    noise of the plane average, and <u'u'> ~ (0.1)^2/3 (uniform noise of amplitude 0.1)."""
    from oracle import stats
    c = cases.channel(96, 32, 64, n_steps=1)
    s = jf.Solver(c, "f64")
    P = stats.profiles(s.jf_plane_sums(s.state(), 1).cpu().numpy())
    y = 0.5 * (c.yf[:-1] + c.yf[1:])
    assert np.max(np.abs(P["u"] - 1.5 * (1 - (y - 1) ** 2))) < 5e-3
    assert np.allclose(P["u'u'"], 0.01 / 3, rtol=0.1) and np.allclose(P["v'v'"], 0.01 / 3, rtol=0.1)
    assert np.max(np.abs(P["u'v'"])) < 5e-4
