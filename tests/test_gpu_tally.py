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


def test_tally_finish_is_the_definition_on_the_same_tables(c1):
    """dw_tally_finish (LCE = detected / generated; line 211: t90) against the oracle's t90_from_hist and a plain
    division ON THE SAME TABLES: LCE exactly (one fp32 rounding of the double quotient), t90 to fp32 rounding."""
    c, ctx, group, comp, K = c1
    n, pps, nb = 200_000 - 7, 33_000, 300
    out = dw.DeviceResults(n, ("flags", "channel", "t", "last_tri"))
    ctx.propagate(dw.DevicePhotons(c.make_photons(n)), c.seed, c.max_steps, out, None)
    ns = -(-n // pps)
    q32 = float(np.float32(0.9))                                                                # the ABI carries the quantile as a float
    for t_min, dt in ((0.0, 1.0), (3.0, 0.37)):                                                 # the second range clamps both ends
        acc = dw.Tally(ns, group, 2, comp, K, nb, t_min, dt)
        ctx.tally(out, n, pps, acc)
        ctx.tally_finish(acc, 0.9)
        torch.cuda.synchronize()
        got = acc.numpy()
        gen = got["fate_by_source"].sum(1).astype(np.float64)
        assert np.array_equal(got["lce"], (got["detected"].astype(np.float64) / gen[:, None]).astype(np.float32))
        for s_ in range(ns):
            want = orc.t90_from_hist(got["time_hist"][s_], t_min, dt, q=q32)
            assert abs(float(got["t90"][s_]) - want) <= 1.5 * float(np.spacing(np.float32(want))), (s_, got["t90"][s_], want)
    # hand-made rows: one bin, an empty row, the crossing exactly on a bin edge, a crossing in the very last (overflow) bin
    rows = np.zeros((5, 40), np.int32)
    rows[0, 7] = 10
    rows[2, 3] = 9; rows[2, 20] = 1                                                             # 0.9 N reached exactly at the end of bin 3
    rows[3, 39] = 5
    rows[4, :] = 3                                                                              # crosses inside the second group of 32 bins
    acc = dw.Tally(5, group, 2, comp, K, 40, 5.0, 2.0)
    acc.time_hist.copy_(torch.from_numpy(rows).to(acc.time_hist.device))
    acc.fate_by_source[:, 1] = 1                                                               # one generated photon per source, none detected
    ctx.tally_finish(acc, 0.9)
    torch.cuda.synchronize()
    got = acc.numpy()
    assert np.all(got["lce"] == 0.0)
    for s_ in (0, 2, 3, 4):
        want = orc.t90_from_hist(rows[s_], 5.0, 2.0, q=q32)
        assert abs(float(got["t90"][s_]) - want) <= 1.5 * float(np.spacing(np.float32(want))), (s_, got["t90"][s_], want)
    assert abs(float(got["t90"][0]) - (5.0 + 2.0 * (7 + 0.9))) < 1e-5                              # all in one bin: linear inside it
    assert math.isnan(float(got["t90"][1]))                                                     # nothing detected
    empty = dw.Tally(2, group, 2, comp, K, 40, 5.0, 2.0)
    ctx.tally_finish(empty, 0.9)
    torch.cuda.synchronize()
    assert np.all(np.isnan(empty.numpy()["lce"]))                                               # nothing generated: 0 / 0
    with pytest.raises(dw.DwError) as ei:
        ctx.tally_finish(acc, 1.5)
    assert ei.value.code == dw.DW_E_ARG


def test_emit_sources_equals_one_emit_per_source(c1):
    """dw_emit_sources (one launch; photon i of source i // pps) against one dw_emit per source with id base s * pps: bit for bit,
    ragged last source, ids beyond 32 bits."""
    c, ctx, _, _, _ = c1
    srcs = [synth.source(synth.SHAPE_POINT, (0.0, 0.0, 100.0)), synth.source_for(1), synth.source_for(4),
            synth.source(synth.SHAPE_BALL, (10.0, -20.0, 300.0), radius=5.0, t_start=2.0, f_singlet=0.22)]
    pps, base = 5_000, (1 << 33) + 17
    n = 4 * pps - 123
    many = ctx.emit_sources(srcs, pps, 77, n=n, id_base=base).numpy()
    for s_, src in enumerate(srcs):
        m = min(pps, n - s_ * pps)
        one = ctx.emit(src, 77, m, id_base=base + s_ * pps).numpy()
        for key in ("pos", "dir", "pol", "wavelength", "t0"):
            assert np.array_equal(many[key][..., s_ * pps:s_ * pps + m], one[key]), (s_, key)
    with pytest.raises(dw.DwError) as ei:
        ctx.emit_sources(srcs, pps, 77, n=4 * pps + 1)
    assert ei.value.code == dw.DW_E_ARG


def _design_study_by_hand(ctx, srcs, pps, seed, max_steps, group, comp, K, nb, dt):
    """The loop dw_design_study runs inside the library, issued call by call: the independent way to the same tables."""
    acc = dw.Tally(len(srcs), group, 2, comp, K, nb, 0.0, dt)
    for s_, src in enumerate(srcs):
        ph = ctx.emit(src, seed, pps, id_base=s_ * pps)
        out = dw.DeviceResults(pps, ("flags", "channel", "t", "last_tri"))
        ctx.propagate(ph, seed, max_steps, out, None)
        ctx.tally(out, pps, pps, acc.view(s_, s_ + 1))
    ctx.tally_finish(acc, 0.9)
    torch.cuda.synchronize()
    return acc.numpy()


def test_design_study_lce_profile_and_t90(c1):
    """Point sources on the axis of the small TPC at five heights (LCE(Z); line 211: t90).  The device pipeline
    against the oracle's own emit -> propagate -> tally, and independence of the batch size."""
    c, ctx, group, comp, K = c1
    zs = [20.0, 120.0, 250.0, 380.0, 480.0]
    srcs = [synth.source(synth.SHAPE_POINT, (0.0, 0.0, z)) for z in zs]
    pps = 100_000
    a = ctx.design_study(srcs, pps, c.seed, c.max_steps, group, 2, comp, K, n_bins=400, dt=1.0, sources_per_batch=2)
    b = ctx.design_study(srcs, pps, c.seed, c.max_steps, group, 2, comp, K, n_bins=400, dt=1.0, sources_per_batch=5)
    h = _design_study_by_hand(ctx, srcs, pps, c.seed, c.max_steps, group, comp, K, 400, 1.0)
    for key in ("detected", "time_hist", "fate_by_source", "absorbed_by_component", "lce", "t90"):
        assert np.array_equal(a[key], b[key]), key                                              # photon ids do not depend on the batching
        assert np.array_equal(a[key], h[key]), key                                              # one call = the loop issued call by call
    assert np.array_equal(a["lce"], (a["detected"] / np.float64(pps)).astype(np.float32))       # PAPER.md line 189, on the device
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
