"""Design variants (synth.config_design; detailed PMTs with a quartz window, a photocathode behind it, a black rim
and a conical PTFE reflector; side walls tiled with 2e4 small sensors) through the C ABI against the oracle, by the criteria of
test_gpu_parity: step-locked identity, statistics (per-channel counts over 2e4 channels, LCE, fates, arrival times), and on the
device the closed form of a photon going straight through a window (tests/test_design_variants.py has it for the oracle)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as orc                       # noqa: E402
from paper_2203_14354_b200 import binding as dw        # noqa: E402
from paper_2203_14354_b200 import synth                # noqa: E402
from test_gpu_parity import check_statistical_parity, gpu_run   # noqa: E402
from test_oracle_pins import photons_from              # noqa: E402

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (run with -m gpu on the B200 box)")


@pytest.mark.parametrize("variant,scale,n", [("both", 1, 200_000), ("detailed_pmt", 2, 100_000), ("side_sensors", 2, 100_000)])
def test_step_locked_parity_on_design_variants(variant, scale, n):
    c = synth.config_design(variant, scale)
    ctx = dw.make_context(c.geometry, c.optics)
    assert ctx.n_chan == c.geometry.n_channels
    o = orc.Oracle(c.geometry, c.optics, bvh=True)
    ph = c.make_photons(n)
    for max_steps in (1, 3):                      # the step counts of test_gpu_parity.test_step_locked_parity
        ref = o.propagate(ph, c.seed, max_steps)
        r = gpu_run(ctx, ph, c.seed, max_steps)
        same = (r["flags"] == ref["flags"]) & (r["steps"] == ref["steps"]) & (r["channel"] == ref["channel"]) & (r["last_tri"] == ref["last_tri"])
        assert same.mean() >= 0.999, f"{variant} x{scale}, {max_steps} steps: identical on {same.mean():.5f}"
        assert np.allclose(r["t"][same], ref["t"][same], rtol=1e-4, atol=1e-4)
        assert ((r["flags"] & dw.H_MEDIUM_MISMATCH) != 0).sum() == 0
        # the literal query (every triangle counts, whatever medium it shows) reports a hit whose near side is not the photon's medium:
        # on a well-formed mesh that only happens through the edge slack at seams
        lit = gpu_run(ctx, ph, c.seed, max_steps, flags=dw.PROP_UNBOUNDED_QUERY)
        assert ((lit["flags"] & dw.H_MEDIUM_MISMATCH) != 0).sum() <= 1e-4 * n
        if max_steps == 3 and variant != "side_sensors":
            assert ((r["flags"] & dw.H_FRESNEL_REFRACT) != 0).sum() > 100          # windows and the liquid surface are in play
    ctx.close()


@pytest.mark.parametrize("variant", ["both", "detailed_pmt"])
def test_statistical_parity_on_design_variants(variant):
    c = synth.config_design(variant, 1)
    ctx = dw.make_context(c.geometry, c.optics)
    res = check_statistical_parity(1, 1_000_000, 1_000_000, ctx=ctx, conf=c)
    assert res["lce_gpu"] > 0.1
    ctx.close()


def test_straight_through_a_pmt_window_on_device():
    """tests/test_design_variants.py::test_straight_through_a_pmt_window_closed_form, on the device."""
    c = synth.config_design("detailed_pmt", 1)
    ctx = dw.make_context(c.geometry, c.optics)
    n = 400_000
    pos = np.tile(np.array([[3.0], [2.0], [100.0]]), (1, n))
    k = np.tile(np.array([[0.0], [0.0], [-1.0]]), (1, n))
    e = np.tile(np.array([[1.0], [0.0], [0.0]]), (1, n))
    ph = photons_from(pos, k, e)
    r1 = gpu_run(ctx, ph, 77, 1)
    refl, refr = (r1["flags"] & dw.H_FRESNEL_REFLECT) != 0, (r1["flags"] & dw.H_FRESNEL_REFRACT) != 0
    p_reach = np.exp(-94.0 / 400.0) * np.exp(-94.0 / 50000.0)
    assert refl.sum() + refr.sum() == pytest.approx(n * p_reach, abs=4 * np.sqrt(n * p_reach * (1 - p_reach)))
    R = ((1.69 - 1.6) / (1.69 + 1.6)) ** 2
    assert abs(refl.sum() - R * (refl.sum() + refr.sum())) < 4 * np.sqrt(R * (refl.sum() + refr.sum()))
    assert np.allclose(r1["z"][refr], 6.0, atol=1e-4)
    r = gpu_run(ctx, ph, 77, 50)
    fl, fate = r["flags"], r["flags"] & 0xF
    other = dw.H_RAYLEIGH | dw.H_REFLECT_DIFFUSE | dw.H_REFLECT_SPECULAR | dw.H_TIR | dw.H_FRESNEL_REFLECT
    through = ((fl & other) == 0) & ((fl & dw.H_FRESNEL_REFRACT) != 0) & (r["steps"] == 2)
    assert through.sum() == refr.sum()
    bulk = (through & (fate == dw.FATE_BULK_ABSORBED)).sum()
    assert abs(bulk - through.sum() * (1 - np.exp(-5.0 / 1000.0))) < 5 * np.sqrt(through.sum() * 0.005)
    at_cathode = through & (fate != dw.FATE_BULK_ABSORBED)
    det = at_cathode & (fate == dw.FATE_DETECTED)
    assert abs(det.sum() - 0.3 * at_cathode.sum()) < 4 * np.sqrt(0.21 * at_cathode.sum())
    assert np.allclose(r["t"][det], (94.0 * 1.69 + 5.0 * 1.6) / 299.792458, rtol=0, atol=2e-5)
    # and photon for photon what the oracle gets with the same draws
    ref = orc.Oracle(c.geometry, c.optics, bvh=True).propagate(ph, 77, 50)
    short = ref["steps"] <= 3
    assert short.mean() > 0.5 and (ref["flags"] == fl)[short].mean() >= 0.999
    ctx.close()
