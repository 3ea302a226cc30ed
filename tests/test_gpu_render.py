"""dw_render (the rendering of the mesh, into device buffers instead of a display) against the
oracle's ray cast: same camera, per pixel the nearest triangle, its distance and the shade.

Criteria: the device forms the pixel directions in single precision, the oracle in double precision rounded to single, so the two
rays of a pixel differ in the last bit and pixels whose ray grazes a triangle edge may resolve differently: ids identical on
>= 99.9 % of the pixels, not counting pixels where the two ids are hit at the same distance (a shared edge: either is right; such
ties must be rare in a generic view); on identical hits the first-hit distance criterion of test_gpu_parity and |shade difference| <= 1 level;
misses are (-1, +inf, 0) on both sides.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as orc                       # noqa: E402
from paper_2203_14354_b200 import binding as dw        # noqa: E402
from paper_2203_14354_b200 import synth                # noqa: E402
from test_gpu_parity import ctx_for, oracle_for, scene_eps   # noqa: E402

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (run with -m gpu on the B200 box)")


def views(g):
    lo, hi = g.xyz.min(0).astype(float), g.xyz.max(0).astype(float)
    mid, size = (lo + hi) / 2, float((hi - lo).max())
    return [
        # inside the liquid, looking up and sideways at the wall and the top array; ragged size (not a multiple of the 16 x 8 tile)
        dict(eye=mid + [0.11 * size, -0.07 * size, -0.2 * size], forward=[0.5, 0.3, 0.8], up=[0.0, 0.0, 1.0], fov_y_deg=70.0, width=203, height=117),
        # from outside, the whole detector in view with background around it
        dict(eye=mid + [1.6 * size, 0.9 * size, 0.7 * size], forward=[-1.6, -0.9, -0.7], up=[0.0, 0.0, 1.0], fov_y_deg=45.0, width=160, height=128),
        # one-pixel-wide and one-pixel-high images
        dict(eye=mid + [0.013 * size, 0.021 * size, 0.0], forward=[0.07, 1.0, 0.1], up=[0.0, 0.0, 1.0], fov_y_deg=30.0, width=1, height=37),
        dict(eye=mid + [0.013 * size, 0.021 * size, 0.0], forward=[1.0, 0.03, -0.1], up=[0.0, 1.0, 0.0], fov_y_deg=120.0, width=41, height=1),
        # on the axis of the detector, rays in the plane x = 0: they run along shared edges of the wall and the fans, where two
        # triangles are hit at the same point and either id is right
        dict(eye=mid, forward=[0.0, 1.0, 0.1], up=[0.0, 0.0, 1.0], fov_y_deg=30.0, width=1, height=37),
    ]


@pytest.mark.parametrize("cfg", [1, 3])
def test_render_against_the_oracle(cfg):
    c, ctx = ctx_for(cfg)
    o = oracle_for(cfg)
    g = c.geometry
    eps = scene_eps(g)
    for k, v in enumerate(views(g)):
        to, do, so = orc.render(o, g, **v)
        tg, dg, sg = (a.cpu().numpy() for a in ctx.render(**v))
        assert tg.shape == (v["height"], v["width"]) and sg.dtype == np.uint8
        same = tg == to
        n_pix = same.size
        # a different id is still right if both sides hit the same point (a shared edge): the distances then agree
        with np.errstate(invalid="ignore"):                 # inf - inf on pixels where both sides miss
            tie = ~same & (tg >= 0) & (to >= 0) & (np.abs(dg.astype(np.float64) - do) <= 1e-5 * do + 16 * eps)
        if k < 4:
            assert tie.sum() <= max(1, int(2e-3 * n_pix)), f"C{cfg} view {k}: {tie.sum()} edge ties in a generic view"
        wrong = ~same & ~tie
        assert wrong.sum() <= max(1, int(1e-3 * n_pix)), f"C{cfg} view {k}: {wrong.sum()} of {n_pix} pixels differ (ids and distances)"
        hit = same & (to >= 0)
        miss = same & (to < 0)
        if k < 2:
            assert hit.sum() > 0.3 * n_pix
        if k == 1:
            assert miss.sum() > 0.2 * n_pix
        assert np.all(np.isinf(dg[miss])) and np.all(sg[miss] == 0)
        # distance: 1e-5 d + eps / |cos(angle to the normal)|, the cosine being what the shade encodes
        cosang = np.maximum(so[hit].astype(float) / 255.0, 1.0 / 255.0)
        err = np.abs(dg[hit].astype(np.float64) - do[hit])
        assert np.all(err <= 1e-5 * do[hit] + 2 * eps / cosang), f"C{cfg} view {k}: worst distance error {err.max()}"
        assert np.all(np.abs(sg[hit].astype(int) - so[hit].astype(int)) <= 1)
        assert (sg[hit] == so[hit]).mean() > 0.98


def test_render_outputs_are_optional_and_errors(tmp_path):
    c, ctx = ctx_for(0)
    g = c.geometry
    v = views(g)[0]
    tri, depth, shade = ctx.render(**v)
    import ctypes as C
    cam = dw.Camera(eye=(C.c_float * 3)(*v["eye"]), forward=(C.c_float * 3)(*v["forward"]), up=(C.c_float * 3)(*v["up"]),
                    fov_y_deg=v["fov_y_deg"], width=v["width"], height=v["height"])
    only = torch.full_like(shade, 7)
    assert ctx.L.dw_render(ctx.h, C.byref(cam), None, None, C.c_void_p(only.data_ptr()), None) == 0
    torch.cuda.synchronize()
    assert torch.equal(only, shade)
    dw.write_pgm(tmp_path / "view.pgm", shade)
    assert (tmp_path / "view.pgm").stat().st_size == len(b"P5\n%d %d\n255\n" % (v["width"], v["height"])) + v["width"] * v["height"]
    for bad in (dict(width=0), dict(height=-3), dict(fov_y_deg=0.0), dict(fov_y_deg=180.0), dict(up=v["forward"]), dict(forward=[0.0, 0.0, 0.0]),
                dict(eye=[float("nan"), 0.0, 0.0]), dict(width=40000)):
        with pytest.raises(dw.DwError) as e:
            ctx.render(**{**v, **bad})
        assert e.value.code == dw.DW_E_ARG, bad
    fresh = dw.Context(0)
    fresh.set_optics(c.optics)
    fresh.set_geometry(g)
    with pytest.raises(dw.DwError) as e:
        fresh.render(**v)
    assert e.value.code == dw.DW_E_STATE
    fresh.close()
