"""dw_design_study_static: the design-study loop with all scratch in the library's fixed device array (no allocation) against the
allocating dw_design_study.  Integer tables: bit for bit; lce / t90 come from the same kernel on equal tables: bit for bit too.
Collected last on purpose (the name sorts after every other test file); passes alone in a fresh process and after the others."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_2203_14354_b200 import binding as dw        # noqa: E402
from paper_2203_14354_b200 import synth                # noqa: E402

pytestmark = pytest.mark.gpu

KEYS = ("detected", "time_hist", "fate_by_source", "absorbed_by_component", "lce", "t90")


@pytest.fixture(scope="module")
def c1():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (run with -m gpu on the B200 box)")
    c = synth.config(1)
    g = c.geometry
    group = np.where(np.arange(g.n_channels) < g.n_channels // 2, 0, 1).astype(np.int32)
    comp = (g.surface + 1).astype(np.int32)
    return c, dw.make_context(g, c.optics), group, comp, int(comp.max()) + 1


def _same(a, b, what):
    for key in KEYS:
        assert np.array_equal(a[key], b[key], equal_nan=key in ("lce", "t90")), (what, key)


def test_static_design_study_equals_the_allocating_one_twice_in_a_row(c1):
    c, ctx, group, comp, K = c1
    srcs = [synth.source(synth.SHAPE_POINT, (0.0, 0.0, z)) for z in (20.0, 120.0, 250.0, 380.0, 480.0)]
    srcs.append(synth.source(synth.SHAPE_BALL, (30.0, -20.0, 300.0), radius=5.0, t_start=2.0, f_singlet=0.22))
    nb, dt = 300, 1.0
    # first call: 6 sources of 60 000 photons = two batches of 4 + 2 sources in the 262 144-photon scratch;
    # second call, straight after it on the same stream: another seed and a size that leaves the first call's photons in the tail
    # of the scratch and makes the batches ragged (7 + 7 + 4 sources of 33 333)
    calls = [(srcs, 60_000, c.seed), (srcs * 3, 33_333, c.seed + 12345)]
    accs = []
    for ss, pps, seed in calls:
        acc = dw.Tally(len(ss), group, 2, comp, K, nb, 0.0, dt)
        accs.append(acc)
    torch.cuda.synchronize()
    free0 = None
    for i, ((ss, pps, seed), acc) in enumerate(zip(calls, accs)):
        if i == 1:
            free0 = torch.cuda.mem_get_info()[0]
        ctx.design_study_static(ss, pps, seed, c.max_steps, acc, 0.9)      # back to back: no synchronisation in between
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                            # the second call took no device memory
    got = [a.numpy() for a in accs]
    for (ss, pps, seed), g_ in zip(calls, got):
        want = ctx.design_study(ss, pps, seed, c.max_steps, group, 2, comp, K, n_bins=nb, dt=dt, sources_per_batch=4)
        _same(g_, want, f"pps {pps}")
        assert np.all(g_["fate_by_source"].sum(1) == pps) and int(g_["detected"].sum()) > 0
    # a third call after the allocating path has run in between: still the same
    acc = dw.Tally(len(srcs), group, 2, comp, K, nb, 0.0, dt)
    ctx.design_study_static(srcs, 60_000, c.seed, c.max_steps, acc, 0.9)
    torch.cuda.synchronize()
    _same(acc.numpy(), got[0], "repeat")


def test_static_design_study_rejects_what_does_not_fit(c1):
    c, ctx, group, comp, K = c1
    src = synth.source(synth.SHAPE_POINT, (0.0, 0.0, 250.0))
    acc = dw.Tally(dw.STATIC_MAX_SOURCES + 1, group, 2, comp, K, 0)
    with pytest.raises(dw.DwError) as ei:
        ctx.design_study_static([src], dw.STATIC_MAX_PHOTONS + 1, 1, c.max_steps, acc)
    assert ei.value.code == dw.DW_E_RANGE and "DW_STATIC_MAX_PHOTONS" in str(ei.value)
    with pytest.raises(dw.DwError) as ei:
        ctx.design_study_static([src] * (dw.STATIC_MAX_SOURCES + 1), 10, 1, c.max_steps, acc)
    assert ei.value.code == dw.DW_E_RANGE and "DW_STATIC_MAX_SOURCES" in str(ei.value)
    with pytest.raises(dw.DwError) as ei:
        ctx.design_study_static([src], 10, 1, c.max_steps, acc, quantile=1.5)
    assert ei.value.code == dw.DW_E_ARG
    torch.cuda.synchronize()
    assert int(acc.numpy()["fate_by_source"].sum()) == 0                    # nothing ran
    # the largest source that fits runs, one source per batch
    acc = dw.Tally(2, group, 2, comp, K, 0)
    ctx.design_study_static([src, src], dw.STATIC_MAX_PHOTONS, 5, c.max_steps, acc)
    torch.cuda.synchronize()
    assert np.all(acc.numpy()["fate_by_source"].sum(1) == dw.STATIC_MAX_PHOTONS)
