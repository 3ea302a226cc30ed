"""GPU parity of dw_tally and the design-study driver.  Integer work: bit-exact against plain counting."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as orc                       # noqa: E402
from paper_2203_14354_b200 import binding as dw        # noqa: E402
from paper_2203_14354_b200 import synth                # noqa: E402
import parity_util as pu                              # noqa: E402

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def c1():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (run with -m gpu on the B200 box)")
    c = synth.config(1)
    g = c.geometry
    group = np.where(np.arange(g.n_channels) < g.n_channels // 2, 0, 1).astype(np.int32)      # channels 0..18 bottom array, 19..37 top
    comp = (g.surface + 1).astype(np.int32)                                                    # component = surface id + 1 (0: no surface)
    return c, dw.make_context(g, c.optics), group, comp, int(comp.max()) + 1


def test_tally_is_plain_counting(c1):
    c, ctx, group, comp, K = c1
    n, pps, nb = 60_000 - 13, 7_000, 64
    ph = c.make_photons(n)
    d = dw.DevicePhotons(ph)
    out = dw.DeviceResults(n, ("flags", "channel", "t", "last_tri"))
    ctx.propagate(d, c.seed, c.max_steps, out, None)
    acc = dw.Tally(-(-n // pps), group, 2, comp, K, nb, 0.0, 2.5)
    ctx.tally(out, n, pps, acc)
    ctx.tally(out, n, pps, acc)                                                                 # accumulates: twice the counts
    torch.cuda.synchronize()
    r, got = out.numpy(), acc.numpy()
    want = orc.tally(r["flags"], r["channel"], r["t"], r["last_tri"], pps, group, 2, comp, K, nb, 0.0, 2.5)
    for key in ("detected", "time_hist", "fate_by_source", "absorbed_by_component"):
        assert np.array_equal(got[key], 2 * want[key]), key
    assert int(got["fate_by_source"].sum()) == 2 * n and got["fate_by_source"][-1].sum() == 2 * (n - (n // pps) * pps)
    assert int(got["absorbed_by_component"].sum()) == 2 * int((r["fate"] == dw.FATE_NAMES.index("surface_absorbed")).sum())
    with pytest.raises(ValueError):
        ctx.tally(out, n, pps // 2, acc)                                                        # more sources than the tables hold
    with pytest.raises(dw.DwError) as ei:
        ctx._check(ctx.L.dw_tally(ctx.h, None, n, pps, None, None))
    assert ei.value.code == dw.DW_E_ARG


def test_design_study_lce_profile_and_t90(c1):
    """Point sources on the axis of the small TPC at five heights (LCE(Z); line 211: t90).  The device pipeline
    against the oracle's own emit -> propagate -> tally, and independence of the batch size."""
    c, ctx, group, comp, K = c1
    zs = [20.0, 120.0, 250.0, 380.0, 480.0]
    srcs = [synth.source(synth.SHAPE_POINT, (0.0, 0.0, z)) for z in zs]
    pps = 100_000
    a = ctx.design_study(srcs, pps, c.seed, c.max_steps, group, 2, comp, K, n_bins=400, dt=1.0, sources_per_batch=2)
    b = ctx.design_study(srcs, pps, c.seed, c.max_steps, group, 2, comp, K, n_bins=400, dt=1.0, sources_per_batch=5)
    for key in ("detected", "time_hist", "fate_by_source", "absorbed_by_component"):
        assert np.array_equal(a[key], b[key]), key                                              # photon ids do not depend on the batching
    assert np.all(a["fate_by_source"].sum(1) == pps)
    o = orc.Oracle(c.geometry, c.optics, bvh=True)
    m = 60_000
    for s, src in enumerate(srcs):
        e = orc.emit(src, c.seed, s * m, m)
        ph = synth.Photons(e["pos"].astype(np.float32), e["dir"].astype(np.float32), e["pol"].astype(np.float32),
                           e["wavelength"].astype(np.float32), e["t0"].astype(np.float32), s * m)
        ref = o.propagate(ph, c.seed, c.max_steps, full=False)
        want = orc.tally(ref["flags"], ref["channel"], ref["t"], ref["last_tri"], m, group, 2, comp, K, 400, 0.0, 1.0)
        for g in range(2):
            pu.assert_binomial_agrees(int(a["detected"][s, g]), pps, int(want["detected"][0, g]), m, 4.0, f"LCE source {s} array {g}")
        t90_o = orc.t90_from_hist(want["time_hist"][0], 0.0, 1.0)
        assert abs(a["t90"][s] - t90_o) < 0.08 * t90_o + 1.0, (a["t90"][s], t90_o)
    lce = a["lce"]
    assert lce[0, 0] > lce[-1, 0] and lce[-1, 1] > lce[0, 1]                                    # the near array sees more
    # the loss table: everything that is not detected, bulk-absorbed or escaped was absorbed on some component
    fb = a["fate_by_source"].sum(0)
    assert int(a["absorbed_by_component"].sum()) == int(fb[dw.FATE_NAMES.index("surface_absorbed")])
    assert a["absorbed_by_component"][0] == 0                                                    # component 0 = triangles without a surface
