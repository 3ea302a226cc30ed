"""Pins of the oracle's ray cast (oracle.camera_rays / oracle.render) against things fixed
outside it: the pinhole projection written the forward way (point -> pixel), and the closed form of a view from inside a box."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2203_14354_b200 import synth


def project(P, eye, forward, up, fov_y_deg, width, height):
    """Textbook look-at + perspective projection, point -> continuous pixel coordinates (pixel centres at integers)."""
    f = np.asarray(forward, float) / np.linalg.norm(forward)
    r = np.cross(f, up)
    r /= np.linalg.norm(r)
    u = np.cross(r, f)
    q = np.asarray(P, float) - np.asarray(eye, float)
    xc, yc, zc = q @ r, q @ u, q @ f                      # camera coordinates: right, up, depth
    t = np.tan(np.radians(fov_y_deg) / 2)
    ndc_x, ndc_y = xc / (zc * t * width / height), yc / (zc * t)
    return (ndc_x + 1) / 2 * width - 0.5, (1 - ndc_y) / 2 * height - 0.5


@pytest.mark.parametrize("w,h,fov", [(7, 5, 50.0), (64, 48, 90.0), (33, 80, 17.5)])
def test_pixel_rays_are_the_inverse_of_the_projection(w, h, fov):
    eye, fwd, up = np.array([3.0, -2.0, 11.0]), np.array([0.3, 1.0, -0.2]), np.array([0.1, 0.0, 1.0])
    d = orc.camera_rays(eye, fwd, up, fov, w, h)
    assert d.shape == (3, w * h) and np.allclose(np.linalg.norm(d, axis=0), 1.0, atol=1e-14)
    for (i, j) in [(0, 0), (w - 1, 0), (0, h - 1), (w - 1, h - 1), (w // 2, h // 3), (w // 3, h - 2)]:
        P = eye + 7.3 * d[:, j * w + i]
        pi, pj = project(P, eye, fwd, up, fov, w, h)
        assert pi == pytest.approx(i, abs=1e-9) and pj == pytest.approx(j, abs=1e-9)
    # orientation: i grows towards forward x up, j grows downwards (against up), the image centre looks along forward
    f = fwd / np.linalg.norm(fwd)
    right = np.cross(f, up)
    assert (d[:, w - 1] - d[:, 0]) @ right > 0 and (d[:, (h - 1) * w] - d[:, 0]) @ up < 0
    if w % 2 and h % 2:
        assert np.allclose(d[:, (h // 2) * w + w // 2], f, atol=1e-15)
    # the vertical field of view: the outermost pixel centres of the middle column are 2 atan((1 - 1/h) tan(fov/2)) apart (odd w)
    if w % 2:
        top, bot = d[:, w // 2], d[:, (h - 1) * w + w // 2]
        assert np.degrees(np.arccos(top @ bot)) == pytest.approx(2 * np.degrees(np.arctan((1 - 1 / h) * np.tan(np.radians(fov) / 2))), abs=1e-9)


def test_view_from_inside_a_box_closed_form():
    """Inside an axis-aligned box the nearest wall along d is the one with the smallest ((d_a > 0 ? hi_a : lo_a) - eye_a) / d_a, the
    shade is |d_a| of that axis, and the triangle is one of the two of that face (synth.box: faces z-, z+, y-, y+, x+, x- in order)."""
    lo, hi = np.array([-40.0, -25.0, 0.0]), np.array([55.0, 30.0, 70.0])
    g = synth.box(lo, hi, 0, 0, 0)
    c = synth.config(0)
    o = orc.Oracle(g, c.optics, bvh=False)
    eye, fwd, up, fov, w, h = np.array([5.0, -3.0, 21.0]), np.array([0.6, 0.5, 0.35]), np.array([0.0, 0.0, 1.0]), 100.0, 96, 64
    tri, dist, shade = orc.render(o, g, eye, fwd, up, fov, w, h)
    d = orc.camera_rays(eye, fwd, up, fov, w, h).astype(np.float32).astype(np.float64)
    tt = np.where(d > 0, (hi - eye)[:, None] / d, (lo - eye)[:, None] / d)
    axis = tt.argmin(axis=0)
    want_t = tt.min(axis=0)
    face = np.where(axis == 2, np.where(d[2] > 0, 1, 0), np.where(axis == 1, np.where(d[1] > 0, 3, 2), np.where(d[0] > 0, 4, 5)))
    sure = np.sort(tt, axis=0)[1] - want_t > 1e-6                        # away from the box edges the wall is unambiguous
    assert sure.mean() > 0.98
    assert np.all(tri.reshape(-1) >= 0)
    assert np.all((tri.reshape(-1) // 2)[sure] == face[sure])
    assert np.allclose(dist.reshape(-1), want_t, rtol=1e-12, atol=1e-9)
    want_shade = np.floor(255.0 * np.abs(d[axis, np.arange(d.shape[1])]) + 0.5)
    assert np.all(np.abs(shade.reshape(-1).astype(int) - want_shade.astype(int))[sure] <= 0)
    # looking away from a box one stands outside of: nothing is hit
    tri, dist, shade = orc.render(o, g, np.array([200.0, 0.0, 30.0]), np.array([1.0, 0.0, 0.0]), up, 60.0, 16, 12)
    assert np.all(tri == -1) and np.all(np.isinf(dist)) and np.all(shade == 0)
    # and towards it: the silhouette of the x+ face (70 high, 55 wide at distance 145) fills the right share of the image
    tri, dist, shade = orc.render(o, g, np.array([200.0, 2.5, 35.0]), np.array([-1.0, 0.0, 0.0]), up, 60.0, 200, 200)
    half = 145.0 * np.tan(np.radians(30.0))
    assert (tri >= 0).mean() == pytest.approx((70.0 * 55.0) / (2 * half) ** 2, rel=0.02)
    assert set(np.unique(tri[tri >= 0]) // 2) == {4} and dist[tri >= 0].min() == pytest.approx(145.0, abs=0.01)   # half a pixel off the axis


def test_write_pgm_round_trip(tmp_path):
    from paper_2203_14354_b200 import binding
    img = (np.arange(5 * 7) * 7 % 256).astype(np.uint8).reshape(5, 7)
    binding.write_pgm(tmp_path / "a.pgm", img)
    raw = (tmp_path / "a.pgm").read_bytes()
    assert raw.startswith(b"P5\n7 5\n255\n") and raw[len(b"P5\n7 5\n255\n"):] == img.tobytes()
