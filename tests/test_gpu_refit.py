"""dw_refit_bvh (geometry variants without a rebuild; the paper's design sweeps move and reshape components of
one detector).  A refit keeps the tree and recomputes every box, so it can only change HOW the nearest hit is found:

  * per-photon outputs and reductions after a refit are bit-identical to those of a fresh build on the moved geometry;
  * first hits after a refit agree with the oracle (brute force over the moved triangles) as a fresh build does;
  * refitting back to the original positions restores the original results;
  * errors: size mismatch, refit before build, a vertex that makes a triangle degenerate or non-finite.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as orc                       # noqa: E402
from paper_2203_14354_b200 import binding as dw        # noqa: E402
from paper_2203_14354_b200 import synth                # noqa: E402
from test_gpu_parity import FULL, gpu_run, scene_eps   # noqa: E402

pytestmark = pytest.mark.gpu

KEYS = FULL + ("chan_count", "time_hist", "fate_count", "total_steps")


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (run with -m gpu on the B200 box)")


@pytest.mark.parametrize("cfg,kind", [(1, "affine"), (1, "component"), (1, "jitter"), (3, "component")])
def test_refit_is_bit_identical_to_a_fresh_build(cfg, kind):
    c = synth.config(cfg)
    g2 = synth.moved(c.geometry, kind)
    n = 150_000 - 7 if cfg == 1 else 60_000
    ph = c.make_photons(n)          # the config's photons: some start outside the moved detector, which is as good a test
    ctx = dw.make_context(c.geometry, c.optics)
    before = gpu_run(ctx, ph, c.seed, c.max_steps, n_bins=100, dt=4.0)
    st = ctx.refit(g2.xyz)
    assert st["n_levels"] == ctx.stats["max_depth"] and st["refit_ms"] > 0.0
    assert np.allclose(st["scene_lo"], g2.xyz.min(0)) and np.allclose(st["scene_hi"], g2.xyz.max(0))
    assert 0 <= st["n_loose_tris"] <= c.geometry.n_tri and 0.5 < st["area_ratio"] < 4.0
    if ctx.stats["grid_res"]:
        assert st["grid_free_cells"] > 0
    after = gpu_run(ctx, ph, c.seed, c.max_steps, n_bins=100, dt=4.0)
    fresh_ctx = dw.make_context(g2, c.optics)
    fresh = gpu_run(fresh_ctx, ph, c.seed, c.max_steps, n_bins=100, dt=4.0)
    for key in KEYS:
        assert np.array_equal(after[key], fresh[key]), f"C{cfg} {kind}: '{key}' after the refit differs from a fresh build"
    assert not np.array_equal(after["t"], before["t"]), "the motion changed nothing: the test has no power"
    # the device-pointer form, and back to the original positions
    back = ctx.refit(torch.from_numpy(c.geometry.xyz).cuda())
    assert back["area_ratio"] == pytest.approx(1.0, abs=1e-6) and back["n_loose_tris"] == 0      # same positions -> same boxes
    again = gpu_run(ctx, ph, c.seed, c.max_steps, n_bins=100, dt=4.0)
    for key in KEYS:
        assert np.array_equal(again[key], before[key]), f"C{cfg} {kind}: '{key}' is not restored by refitting back"
    ctx.close(); fresh_ctx.close()


def test_first_hit_after_refit_against_the_oracle():
    """Criterion of test_gpu_parity.check_first_hit on the moved geometry, the oracle searching all triangles one by one."""
    c = synth.config(1)
    g2 = synth.moved(c.geometry, "affine")
    ctx = dw.make_context(c.geometry, c.optics)
    ctx.refit(g2.xyz)
    o = orc.Oracle(g2, c.optics, bvh=False)
    rng = np.random.default_rng(11)
    n = 4000
    lo, hi = g2.xyz.min(0).astype(np.float64), g2.xyz.max(0).astype(np.float64)
    origin = (lo + (hi - lo) * rng.uniform(0.2, 0.8, (n, 3))).T.astype(np.float32).copy()
    d = rng.normal(size=(3, n))
    d = (d / np.linalg.norm(d, axis=0)).astype(np.float32)
    to, do = o.first_hit(origin, d, exclude=None, use_bvh=False)
    tg, dg = ctx.first_hit(torch.from_numpy(origin).cuda(), torch.from_numpy(d).cuda(), None)
    tg, dg = tg.cpu().numpy(), dg.cpu().numpy().astype(np.float64)
    same = tg == to
    assert same.mean() >= 0.9999
    hit = same & (to >= 0)
    assert hit.sum() > n // 2
    assert np.quantile(np.abs(dg[hit] - do[hit]) / (1e-5 * do[hit] + scene_eps(g2)), 0.99) <= 1.0
    ctx.close()


def test_refit_errors():
    c = synth.config(0)
    ctx = dw.Context(0)
    ctx.set_optics(c.optics)
    ctx.set_geometry(c.geometry)
    with pytest.raises(dw.DwError) as e:
        ctx.refit(c.geometry.xyz)
    assert e.value.code == dw.DW_E_STATE
    ctx.build_bvh()
    with pytest.raises(dw.DwError) as e:
        ctx.refit(c.geometry.xyz[:-1])
    assert e.value.code == dw.DW_E_ARG
    ctx.refit(c.geometry.xyz)                      # unchanged positions: fine
    bad = c.geometry.xyz.copy()
    i0, i1 = c.geometry.idx[0, 0], c.geometry.idx[0, 1]
    bad[i1] = bad[i0]                              # triangle 0 collapses to a segment
    with pytest.raises(dw.DwError) as e:
        ctx.refit(bad)
    assert e.value.code == dw.DW_E_RANGE and "zero area" in str(e.value)
    with pytest.raises(dw.DwError) as e:           # the context lost its geometry and its tree: nothing runs on a half-updated state
        ctx.refit(c.geometry.xyz)
    assert e.value.code == dw.DW_E_STATE
    ctx.set_geometry(c.geometry)
    ctx.build_bvh()
    bad = c.geometry.xyz.copy()
    bad[c.geometry.idx[0, 2], 1] = np.nan
    with pytest.raises(dw.DwError) as e:
        ctx.refit(bad)
    assert e.value.code == dw.DW_E_RANGE
    ctx.close()
