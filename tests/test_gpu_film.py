"""GPU parity of thin-film surfaces against the oracle and against the closed forms the oracle is pinned to."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as orc                       # noqa: E402
from paper_2203_14354_b200 import binding as dw        # noqa: E402
from paper_2203_14354_b200 import synth                # noqa: E402
import parity_util as pu                              # noqa: E402
from test_oracle_film import film_column               # noqa: E402
from test_gpu_parity import gpu_run, check_statistical_parity, FULL   # noqa: E402

pytestmark = pytest.mark.gpu


def beam(n, theta_deg=0.0, x0=0.0, pol="s"):
    th = math.radians(theta_deg)
    pos = np.repeat(np.array([[x0], [0.0], [50.0]]), n, 1)
    k = np.repeat(np.array([[math.sin(th)], [0.0], [math.cos(th)]]), n, 1)
    ev = {"s": [0.0, 1.0, 0.0], "p": [math.cos(th), 0.0, -math.sin(th)], "m": [math.cos(th) / math.sqrt(2), 1 / math.sqrt(2), -math.sin(th) / math.sqrt(2)]}[pol]
    e = np.repeat(np.array(ev)[:, None], n, 1)
    return synth.Photons(pos.astype(np.float32), k.astype(np.float32), e.astype(np.float32), np.full(n, 175.0, np.float32), np.zeros(n, np.float32))


@pytest.mark.parametrize("case", [(1.6, 0.81, 1.86, 3000.0, 0.25, 0.0, "s"), (1.0, 1.3, 0.7, 0.0, 1.0, 0.0, "s"), (1.2, math.sqrt(1.69 * 1.2), 0.0, 175.0 / (4 * math.sqrt(1.69 * 1.2)), 1.0, 0.0, "s"),
                                  (1.6, 0.81, 1.86, 15.0, 0.5, 25.0, "s"), (1.6, 0.81, 1.86, 15.0, 0.5, 25.0, "p"), (1.6, 1.38, 0.02, 40.0, 0.5, 20.0, "m"), (1.0, 1.4, 0.0, 50.0, 1.0, 30.0, "m")])
def test_film_column_on_device(case):
    """Fractions reflected / transmitted / detected-in-the-film against the closed forms (thick silicon 0.43606, bare interface
    0.065795, perfect anti-reflection 0) and against the oracle's coefficients, and photon by photon against the oracle."""
    n3, nf, kf, d, det, theta, pol = case
    g, op = film_column(n3, nf, kf, d, det)
    ctx = dw.make_context(g, op)
    n = 200_000
    ph = beam(n, theta, -75.0 * math.tan(math.radians(theta)), pol)     # up 50 mm, back down 100 mm: centre the path on the +-50 mm sheets
    r = gpu_run(ctx, ph, 9, 20)
    ref = orc.Oracle(g, op, bvh=False).propagate(ph, 9, 20)
    same = (r["flags"] == ref["flags"]) & (r["channel"] == ref["channel"]) & (r["steps"] == ref["steps"])
    assert same.mean() >= 0.9995, f"identical on {same.mean():.5f}"
    assert int(r["fate_count"][dw.FATE_NAMES.index("escaped")]) == 0 and np.all((r["flags"] & dw.H_FILM) != 0)
    Rs, Rp, Ts, Tp = orc.film_coefficients(1.69, nf, kf, d, n3, 175.0, math.cos(math.radians(theta)))
    w = {"s": (1.0, 0.0), "p": (0.0, 1.0), "m": (0.5, 0.5)}[pol]
    R, T = w[0] * Rs + w[1] * Rp, w[0] * Ts + w[1] * Tp
    if n1_total_reflection(theta, n3):
        assert T == 0
    c = r["chan_count"].astype(float) / n
    sig = lambda p: 4 * math.sqrt(max(p * (1 - p), 1e-9) / n) + 2e-5
    assert abs(c[0] - R) < sig(R) and abs(c[1] - T) < sig(T) and abs(c[2] - det * (1 - R - T)) < sig(det * (1 - R - T))
    k = np.stack([r["kx"], r["ky"], r["kz"]])
    assert np.abs(k[:, same] - ref["dir"][:, same]).max() < 2e-5
    ctx.close()


def n1_total_reflection(theta_deg, n3):
    return 1.69 * math.sin(math.radians(theta_deg)) / n3 >= 1.0


_FILM_C1 = {}


def c1_with_silicon_cathodes():
    if not _FILM_C1:
        base = synth.config(1)
        op = synth.with_film(base.optics, synth.SURF_CATHODE, 0.81, 1.86, 100.0, detect=0.5)    # Table 8 silicon, opaque at 100 nm
        conf = synth.Config(base.name + " (silicon film cathodes)", base.geometry, op, base.n_photons, base.seed, base.max_steps, base.make_photons)
        _FILM_C1["x"] = (conf, dw.make_context(conf.geometry, conf.optics))
    return _FILM_C1["x"]


def test_film_step_locked_and_scheduler_identity_on_c1():
    conf, ctx = c1_with_silicon_cathodes()
    n = 200_000
    ph = conf.make_photons(n)
    ref = orc.Oracle(conf.geometry, conf.optics, bvh=True).propagate(ph, conf.seed, 3)
    r = gpu_run(ctx, ph, conf.seed, 3)
    same = (r["flags"] == ref["flags"]) & (r["steps"] == ref["steps"]) & (r["channel"] == ref["channel"]) & (r["last_tri"] == ref["last_tri"])
    assert same.mean() >= 0.999 and ((r["flags"] & dw.H_FILM) != 0).sum() > 1000
    a = gpu_run(ctx, ph, conf.seed, conf.max_steps, n_bins=100, dt=4.0)
    b = gpu_run(ctx, ph, conf.seed, conf.max_steps, n_bins=100, dt=4.0, flags=dw.PROP_LEGACY_SCHEDULER)
    for key in FULL + ("chan_count", "time_hist", "fate_count", "total_steps"):
        assert np.array_equal(a[key], b[key]), key


def test_film_statistical_parity_on_c1():
    conf, ctx = c1_with_silicon_cathodes()
    check_statistical_parity(1, 1_000_000, 1_000_000, ctx=ctx, conf=conf)


def test_set_films_argument_checks():
    c = synth.config(1)
    ctx = dw.Context(0)
    with pytest.raises(dw.DwError) as ei:
        ctx.set_films(np.zeros(4, np.int32), np.ones((4, 1)), np.zeros((4, 1)), np.zeros((4, 1)), 175.0, 1.0)
    assert ei.value.code == dw.DW_E_STATE
    ctx.set_optics(c.optics)
    S = c.optics.detect.shape[0]
    on = np.zeros(S, np.int32); on[1] = 1
    with pytest.raises(dw.DwError) as ei:                      # wrong grid
        ctx.set_films(on, np.ones((S, 2)), np.zeros((S, 2)), np.zeros((S, 2)), 175.0, 1.0)
    assert ei.value.code == dw.DW_E_ARG
    for bad in (dict(n=-1.0), dict(k=-0.1), dict(d=-5.0), dict(n=float("nan"))):
        fn, fk, fd = np.ones((S, 1)), np.zeros((S, 1)), np.zeros((S, 1))
        fn[1] = bad.get("n", 1.0); fk[1] = bad.get("k", 0.0); fd[1] = bad.get("d", 0.0)
        with pytest.raises(dw.DwError) as ei:
            ctx.set_films(on, fn, fk, fd, c.optics.lambda0, c.optics.dlambda)
        assert ei.value.code == dw.DW_E_RANGE, bad
    ctx.set_films(on, np.ones((S, 1)), np.zeros((S, 1)), np.zeros((S, 1)), c.optics.lambda0, c.optics.dlambda)
    ctx.set_films(None, None, None, None, 0.0, 1.0)            # removes them
    ctx.close()
