"""GPU parity of dw_emit against the oracle's emission, same seeds, same Philox draws.

Tolerances (fp32 kernel against the fp64 oracle, derived from the arithmetic): every quantity is a short chain of correctly
rounded or <= 2 ulp operations (sqrt, cbrt, sincospi, log) on exactly shared uniforms, so the relative error is a few 2^-24:
positions 4e-7 x scale, unit vectors 1e-6 (the polarisation divides by |k x r|, so its error grows as 1/|k x r|), wavelength and
time 4e-6 relative to their magnitude.  The singlet / triplet branch is an integer decision taken in fp32 on both sides."""
import math

import numpy as np
import pytest
from scipy import stats

torch = pytest.importorskip("torch")

from oracle import oracle as orc                       # noqa: E402
from paper_2203_14354_b200 import binding as dw        # noqa: E402
from paper_2203_14354_b200 import synth                # noqa: E402
import parity_util as pu                              # noqa: E402

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (run with -m gpu on the B200 box)")
    c = synth.config(1)
    return c, dw.make_context(c.geometry, c.optics)


SOURCES = {
    "cylinder": synth.source_for(2),
    "ball": synth.source_for(4),
    "point": synth.source(synth.SHAPE_POINT, (1.5, -2.5, 3.5), f_singlet=0.22, t_start=5.0),
    "mono": synth.source(synth.SHAPE_CYLINDER, (3.0, 4.0, 0.0), 249.0, 2.0, 494.0, lambda_mean=175.0, lambda_fwhm=0.0, tau1=0.0, tau3=0.0),
}


@pytest.mark.parametrize("name", list(SOURCES))
def test_emit_matches_the_oracle_photon_by_photon(ctx, name):
    _, c = ctx
    src, n, seed, base = SOURCES[name], 300_000 - 7, 31, (1 << 33) + 12345          # ragged n, ids beyond 32 bits
    g = c.emit(src, seed, n, id_base=base).numpy()
    o = orc.emit(src, seed, base, n)
    scale = max(1.0, float(np.abs(o["pos"]).max()))
    assert np.abs(g["pos"] - o["pos"]).max() <= 4e-7 * scale + 1e-6
    assert np.abs(g["dir"] - o["dir"]).max() <= 1e-6
    # e = (k x r) / |k x r|: an error of ~1e-7 in k x r becomes 1e-7 / |k x r| in e.  P(|k x r| < s) = s^2 / 2, so all but 0.1 % of
    # the photons have |k x r| > 0.045 (error < 1e-5) and the smallest of 3e5 is ~2.6e-3 (error ~1e-4)
    err_e = np.abs(g["pol"] - o["pol"]).max(0)
    assert np.quantile(err_e, 0.999) <= 2e-5 and err_e.max() <= 5e-3
    assert np.abs((g["pol"].astype(np.float64) * g["dir"]).sum(0)).max() <= 2e-6
    assert np.abs((g["pol"].astype(np.float64) ** 2).sum(0) - 1).max() <= 2e-6
    assert np.abs(g["wavelength"] - o["wavelength"]).max() <= 4e-6 * 200.0
    # the branch (tau_1 or tau_3) is the same on both sides, so the times agree to rounding everywhere
    assert np.all(np.abs(g["t0"] - o["t0"]) <= 4e-6 * np.maximum(np.abs(o["t0"]), 1.0))


def test_emit_laws_on_the_device_output(ctx):
    _, c = ctx
    n = 400_000
    g = c.emit(synth.source_for(2), 41, n).numpy()
    x, y, z = g["pos"].astype(np.float64)
    assert stats.kstest((x * x + y * y) / 1299.0 ** 2, "uniform").pvalue > 1e-4
    assert stats.kstest((z - 2.0) / 2597.0, "uniform").pvalue > 1e-4
    assert stats.kstest((g["dir"][2].astype(np.float64) + 1) / 2, "uniform").pvalue > 1e-4
    sigma = 10.2 / (2 * math.sqrt(2 * math.log(2)))
    assert stats.kstest(g["wavelength"].astype(np.float64), stats.norm(174.8, sigma).cdf).pvalue > 1e-4
    cdf = lambda t: 0.66 * (1 - np.exp(-t / 3.5)) + 0.34 * (1 - np.exp(-t / 24.0))
    assert stats.kstest(g["t0"].astype(np.float64), cdf).pvalue > 1e-4


def test_emit_depends_on_seed_and_photon_id_only(ctx):
    _, c = ctx
    src = synth.source_for(2)
    whole = c.emit(src, 51, 50_000, id_base=1000).numpy()
    part = c.emit(src, 51, 10_000, id_base=21_000).numpy()
    for key in ("pos", "dir", "pol", "wavelength", "t0"):
        assert np.array_equal(whole[key][..., 20_000:30_000], part[key])
    again = c.emit(src, 51, 50_000, id_base=1000).numpy()
    assert all(np.array_equal(whole[k], again[k]) for k in whole)
    assert c.emit(src, 51, 0).n == 0                                              # empty batch


def test_emit_rejects_bad_sources(ctx):
    _, c = ctx
    for bad in (dict(shape=3), dict(radius=-1.0), dict(lambda_sigma=-0.1), dict(tau1=-1.0), dict(f_singlet=1.5), dict(z0=5.0, z1=1.0),
                dict(radius=float("nan"))):
        src = dict(synth.source_for(1), **bad)
        with pytest.raises(dw.DwError) as ei:
            c.emit(src, 1, 10)
        assert ei.value.code == dw.DW_E_ARG, bad


def test_emit_then_propagate_agrees_with_the_oracle_pipeline(ctx):
    """The emitted batch goes straight to dw_propagate; the oracle does the same with its own emission.  Same seeds; the
    fp32 / fp64 photons differ in the last bits, so the comparison is statistical (BASELINE.json: LCE within 0.2 % absolute,
    per-channel 4 sigma, arrival times KS p > 0.01)."""
    cfg, c = ctx
    n, seed = 600_000, cfg.seed
    src = synth.source_for(1)
    d = c.emit(src, seed, n)
    out = dw.DeviceResults(n, ("flags", "channel", "t", "steps"))
    hist = dw.DeviceHists(c.n_chan, 0, 0.0, 1.0)
    c.propagate(d, seed, cfg.max_steps, out, hist)
    torch.cuda.synchronize()
    r, h = out.numpy(), hist.numpy()
    assert int(h["fate_count"].sum()) == n
    m = 300_000
    e = orc.emit(src, seed, 0, m)
    ph = synth.Photons(e["pos"].astype(np.float32), e["dir"].astype(np.float32), e["pol"].astype(np.float32),
                       e["wavelength"].astype(np.float32), e["t0"].astype(np.float32), 0)
    ref = orc.Oracle(cfg.geometry, cfg.optics, bvh=True).propagate(ph, seed, cfg.max_steps, full=True)
    pu.assert_fraction_agrees(int(h["fate_count"][0]), n, int(ref["fate_count"][0]), m, 2e-3, "LCE after device emission")
    pu.assert_channels_agree(h["chan_count"], n, ref["chan_count"], m, "per-channel after device emission")
    tg = r["t"][(r["flags"] & 0xF) == 0]
    to = ref["t"][(ref["flags"] & 0xF) == 0]
    assert pu.ks_pvalue(tg, to) > 0.01
    # the scintillation delay is in the arrival times: mean detected time exceeds the prompt-only transit by about <t0>
    assert tg.mean() > 0.66 * 3.5 + 0.34 * 24.0
