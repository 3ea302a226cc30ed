"""Pins of the oracle's thin-film surface.

PAPER.md line 175: surface reflectivity "calculated using Fresnel equations from the specified complex index of refraction and
surface thickness"; Table 8 (lines 356-357): silicon n = 0.81, k = 1.86.  The oracle uses the Airy summation; the pins are closed
forms of thin-film optics and an independent characteristic-matrix computation."""
import math

import numpy as np

from oracle import oracle as orc

N_LXE, N_GXE, N_QUARTZ = 1.69, 1.0, 1.60


def bare(n1, n2, c1):
    """Fresnel intensity coefficients of a single interface between real indices (textbook sine / tangent forms)."""
    t1 = math.acos(c1)
    t2 = math.asin(n1 * math.sin(t1) / n2)
    if t1 == 0.0:
        r = ((n1 - n2) / (n1 + n2)) ** 2
        return r, r
    return (math.sin(t1 - t2) / math.sin(t1 + t2)) ** 2, (math.tan(t1 - t2) / math.tan(t1 + t2)) ** 2


def matrix_method(n1, nf, kf, d, n3, lam, c1):
    """Characteristic matrix of one layer (Born & Wolf / Macleod): tilted admittances eta = n cos (s) or n / cos (p)."""
    n2 = complex(nf, kf)
    s1 = math.sqrt(1 - c1 * c1)
    c2 = np.sqrt(1 - (n1 * s1 / n2) ** 2 + 0j)
    if (n2 * c2).imag < 0:
        c2 = -c2
    s3 = n1 * s1 / n3
    c3 = complex(math.sqrt(1 - s3 * s3), 0) if s3 < 1 else complex(0, math.sqrt(s3 * s3 - 1))
    delta = 2 * math.pi * d * n2 * c2 / lam
    out = []
    for pol in "sp":
        eta = (lambda n, c: n * c) if pol == "s" else (lambda n, c: n / c)
        e1, e2, e3 = eta(n1, c1), eta(n2, c2), eta(n3, c3)
        m11, m12, m21, m22 = np.cos(delta), -1j * np.sin(delta) / e2, -1j * e2 * np.sin(delta), np.cos(delta)
        B, Cc = m11 + m12 * e3, m21 + m22 * e3
        r = (e1 * B - Cc) / (e1 * B + Cc)
        R = abs(r) ** 2
        T = 4 * e1.real * e3.real / abs(e1 * B + Cc) ** 2 if s3 < 1 else 0.0
        out.append((R, T))
    return out[0][0], out[1][0], out[0][1], out[1][1]


def test_zero_thickness_is_the_bare_interface():
    for n1, n3 in ((N_LXE, N_GXE), (N_GXE, N_LXE), (N_LXE, N_QUARTZ)):
        for deg in (0.0, 10.0, 20.0, 30.0, 35.0):
            c1 = math.cos(math.radians(deg))
            if n1 * math.sin(math.radians(deg)) / n3 >= 1:
                continue
            Rs, Rp, Ts, Tp = orc.film_coefficients(n1, 1.37, 0.4, 0.0, n3, 175.0, c1)     # whatever the film is made of
            bs, bp = bare(n1, n3, c1)
            assert abs(Rs - bs) < 1e-12 and abs(Rp - bp) < 1e-12
            assert abs(Rs + Ts - 1) < 1e-12 and abs(Rp + Tp - 1) < 1e-12
    Rs, Rp, _, _ = orc.film_coefficients(N_LXE, 1.2, 0.0, 0.0, N_GXE, 175.0, math.cos(math.radians(20.0)))
    assert abs(Rs - 0.103131) < 1e-6 and abs(Rp - 0.035908) < 1e-6


def test_lossless_film_conserves_energy_and_has_the_quarter_and_half_wave_values():
    rng = np.random.default_rng(3)
    for _ in range(200):
        n1, nf, n3 = rng.uniform(1.0, 2.0, 3)
        d, lam, c1 = rng.uniform(0, 400), rng.uniform(160, 190), rng.uniform(0.05, 1.0)
        Rs, Rp, Ts, Tp = orc.film_coefficients(n1, nf, 0.0, d, n3, lam, c1)
        if n1 * math.sqrt(1 - c1 * c1) / n3 < 1 and n1 * math.sqrt(1 - c1 * c1) / nf < 1:
            assert abs(Rs + Ts - 1) < 1e-10 and abs(Rp + Tp - 1) < 1e-10
    n1, nf, n3, lam = 1.0, 1.38, N_LXE, 175.0                                                # MgF2-like layer on LXe, from vacuum
    R, _, T, _ = orc.film_coefficients(n1, nf, 0.0, lam / (4 * nf), n3, lam, 1.0)
    assert abs(R - ((n1 * n3 - nf * nf) / (n1 * n3 + nf * nf)) ** 2) < 1e-12 and abs(R + T - 1) < 1e-12
    R, _, _, _ = orc.film_coefficients(n1, nf, 0.0, lam / (2 * nf), n3, lam, 1.0)
    assert abs(R - ((n1 - n3) / (n1 + n3)) ** 2) < 1e-12                                      # a half-wave layer is absent
    R, _, _, _ = orc.film_coefficients(1.0, math.sqrt(N_LXE), 0.0, lam / (4 * math.sqrt(N_LXE)), N_LXE, lam, 1.0)
    assert R < 1e-24                                                                          # perfect anti-reflection


def test_thick_absorbing_film_is_its_front_face():
    """Table 8 silicon (0.81, 1.86): opaque after a few hundred nm; R = |(n1 - n2) / (n1 + n2)|^2 at normal incidence."""
    for n1 in (N_GXE, N_LXE):
        expect = ((n1 - 0.81) ** 2 + 1.86 ** 2) / ((n1 + 0.81) ** 2 + 1.86 ** 2)
        for n3 in (1.0, 1.6, 3.0):
            Rs, Rp, Ts, Tp = orc.film_coefficients(n1, 0.81, 1.86, 3000.0, n3, 175.0, 1.0)
            assert abs(Rs - expect) < 1e-9 and abs(Rp - expect) < 1e-9 and Ts < 1e-50 and Tp < 1e-50
    assert abs(((N_LXE - 0.81) ** 2 + 1.86 ** 2) / ((N_LXE + 0.81) ** 2 + 1.86 ** 2) - 0.43606) < 1e-5
    # absorbing film: something is always lost, and grazing incidence reflects everything
    Rs, Rp, Ts, Tp = orc.film_coefficients(N_LXE, 0.81, 1.86, 20.0, 1.0, 175.0, 0.7)
    assert 0 < 1 - Rs - Ts < 1 and 0 < 1 - Rp - Tp < 1
    Rs, Rp, _, _ = orc.film_coefficients(N_LXE, 0.81, 1.86, 20.0, 1.0, 175.0, 1e-6)
    assert Rs > 0.9999 and Rp > 0.9999


def test_evanescent_exit_and_frustrated_total_reflection():
    c1 = math.cos(math.radians(60.0))                           # beyond the LXe -> GXe critical angle of 36.3 deg
    Rs, Rp, Ts, Tp = orc.film_coefficients(N_LXE, 1.4, 0.0, 50.0, N_GXE, 175.0, c1)
    assert Ts == 0 and Tp == 0 and abs(Rs - 1) < 1e-12 and abs(Rp - 1) < 1e-12              # lossless: all reflected
    # a thin gas gap between two liquids lets light tunnel; a thick one does not
    thin = orc.film_coefficients(N_LXE, 1.0, 0.0, 10.0, N_LXE, 175.0, c1)
    thick = orc.film_coefficients(N_LXE, 1.0, 0.0, 2000.0, N_LXE, 175.0, c1)
    assert thin[2] > 0.5 and abs(thin[0] + thin[2] - 1) < 1e-10 and thick[2] < 1e-20 and abs(thick[0] - 1) < 1e-12


def test_airy_summation_equals_the_characteristic_matrix():
    rng = np.random.default_rng(9)
    for _ in range(500):
        n1, n3 = rng.uniform(1.0, 2.0, 2)
        nf, kf = rng.uniform(0.3, 2.5), rng.uniform(0.0, 2.5)
        d, lam, c1 = rng.uniform(0, 300), rng.uniform(160, 190), rng.uniform(0.05, 1.0)
        got = orc.film_coefficients(n1, nf, kf, d, n3, lam, c1)
        want = matrix_method(n1, nf, kf, d, n3, lam, c1)
        assert np.allclose(got, want, rtol=1e-9, atol=1e-12), (n1, nf, kf, d, n3, lam, c1, got, want)
        assert all(-1e-12 <= v <= 1 + 1e-12 for v in got) and got[0] + got[2] <= 1 + 1e-10 and got[1] + got[3] <= 1 + 1e-10


def test_film_event_outcomes_and_state():
    nhat = np.array([0.0, 0.0, -1.0])                            # photon travels towards +z, the facing normal points back
    th = math.radians(25.0)
    k = np.array([math.sin(th), 0.0, math.cos(th)])
    e = np.array([0.0, 1.0, 0.0])                                # s-polarised
    Rs, Rp, Ts, Tp = orc.film_coefficients(N_LXE, 0.81, 1.86, 15.0, N_QUARTZ, 175.0, math.cos(th))
    oc, k2, e2, R, T = orc.film(N_LXE, 0.81, 1.86, 15.0, N_QUARTZ, 175.0, nhat, k, e, 0.5 * Rs)
    assert oc == 0 and abs(R - Rs) < 1e-12 and abs(T - Ts) < 1e-12
    assert np.allclose(k2, [math.sin(th), 0.0, -math.cos(th)]) and abs(abs(e2[1]) - 1) < 1e-12       # mirror, s stays s
    oc, k2, e2, _, _ = orc.film(N_LXE, 0.81, 1.86, 15.0, N_QUARTZ, 175.0, nhat, k, e, Rs + 0.5 * Ts)
    assert oc == 1 and abs(N_LXE * math.sin(th) - N_QUARTZ * math.hypot(k2[0], k2[1])) < 1e-12        # Snell into medium 3
    assert abs(k2 @ e2) < 1e-12 and abs(e2 @ e2 - 1) < 1e-12
    oc, k2, e2, _, _ = orc.film(N_LXE, 0.81, 1.86, 15.0, N_QUARTZ, 175.0, nhat, k, e, Rs + Ts + 0.5 * (1 - Rs - Ts))
    assert oc == 2 and np.array_equal(k2, k) and np.array_equal(e2, e)                                 # absorbed: state untouched
    ep = np.array([math.cos(th), 0.0, -math.sin(th)])            # p-polarised
    _, _, _, R, T = orc.film(N_LXE, 0.81, 1.86, 15.0, N_QUARTZ, 175.0, nhat, k, ep, 2.0)
    assert abs(R - Rp) < 1e-12 and abs(T - Tp) < 1e-12
    em = (e + ep) / math.sqrt(2.0)                               # mixed: intensities add (S8)
    _, _, _, R, T = orc.film(N_LXE, 0.81, 1.86, 15.0, N_QUARTZ, 175.0, nhat, k, em, 2.0)
    assert abs(R - 0.5 * (Rs + Rp)) < 1e-12 and abs(T - 0.5 * (Ts + Tp)) < 1e-12
    oc, k2, e2, R, _ = orc.film(N_LXE, 0.81, 1.86, 3000.0, 1.0, 175.0, nhat, np.array([0.0, 0.0, 1.0]), e, 0.1)
    assert oc == 0 and np.allclose(k2, [0, 0, -1]) and abs(R - 0.43606) < 1e-5                         # normal incidence never aborts


# ----------------------------------------------------------------------------- the film inside the propagation loop
from paper_2203_14354_b200 import synth          # noqa: E402


def film_column(n_behind, nf, kf, d_nm, detect):
    """Column: perfect detector ch 0 at z = 0, film sheet (ch 2) at z = 100 between LXe below and material 3 above, perfect detector
    ch 1 at z = 110.  Materials: 0 LXe 1.69, 1 GXe 1.0, 2 solid, 3 'behind' (index n_behind).  No bulk processes."""
    A = (-50.0, 50.0)

    def sheet(z, mi, mo, surf, ch):
        xyz = np.array([[A[0], A[0], z], [A[1], A[0], z], [A[1], A[1], z], [A[0], A[1], z]], np.float32)
        return synth.Geometry(xyz, np.array([[0, 1, 2], [0, 2, 3]], np.int32), np.full(2, mi, np.int32), np.full(2, mo, np.int32),
                              np.full(2, surf, np.int32), np.full(2, ch, np.int32), max(ch + 1, 0))
    g = synth.merge(sheet(0.0, 2, 0, 0, 0), sheet(100.0, 0, 3, 1, 2), sheet(110.0, 3, 2, 0, 1))   # normals +z: inner below, outer above
    g.n_channels = 3
    f = lambda v: np.asarray(v, np.float32)[:, None].copy()
    inf = np.inf
    op = synth.Optics(1, 175.0, 1.0, f([1.69, 1.0, 1.0, n_behind]), f([inf] * 4), f([inf] * 4),
                      f([1.0, detect]), f([0, 0]), f([0, 0]), f([0, 0]))                           # surface 0 perfect detector, 1 the film
    return g, synth.with_film(op, 1, nf, kf, d_nm)


def shoot(g, op, n, theta_deg=0.0, seed=1, x0=0.0):
    th = math.radians(theta_deg)
    pos = np.repeat(np.array([[x0], [0.0], [50.0]]), n, 1)
    k = np.repeat(np.array([[math.sin(th)], [0.0], [math.cos(th)]]), n, 1)
    e = np.repeat(np.array([[0.0], [1.0], [0.0]]), n, 1)                                          # s-polarised
    ph = synth.Photons(pos.astype(np.float32), k.astype(np.float32), e.astype(np.float32), np.full(n, 175.0, np.float32),
                       np.zeros(n, np.float32))
    return orc.Oracle(g, op, bvh=False).propagate(ph, seed, 20)


def test_film_in_the_propagation_loop_against_closed_forms():
    n = 200_000
    sig = lambda p: 4 * math.sqrt(max(p * (1 - p), 1e-9) / n) + 1e-12
    # thick silicon (Table 8) seen from LXe: R = 0.43606, T = 0, the rest is absorbed and detected with probability 0.25
    out = shoot(*film_column(1.6, 0.81, 1.86, 3000.0, 0.25), n)
    c = out["chan_count"].astype(float) / n
    R = ((1.69 - 0.81) ** 2 + 1.86 ** 2) / ((1.69 + 0.81) ** 2 + 1.86 ** 2)
    assert abs(c[0] - R) < sig(R) and c[1] == 0
    assert abs(c[2] - 0.25 * (1 - R)) < sig(0.25 * (1 - R))
    assert int(out["fate_count"][orc.FATE_SURFACE_ABSORBED]) == n - int(out["chan_count"].sum())
    assert np.all((out["flags"] & orc.H_FILM) != 0)
    assert np.all(((out["flags"] & orc.H_REFLECT_SPECULAR) != 0) == (out["channel"] == 0))
    # zero thickness between LXe and GXe: the bare interface, 6.5795 % reflected (paper: 6.5 %), nothing absorbed
    out = shoot(*film_column(1.0, 1.3, 0.7, 0.0, 1.0), n, seed=2)
    c = out["chan_count"].astype(float) / n
    R = ((1.69 - 1.0) / (1.69 + 1.0)) ** 2
    assert abs(R - 0.065795) < 1e-6 and abs(c[0] - R) < sig(R) and c[2] == 0 and abs(c[0] + c[1] - 1) < 1e-12
    # perfect anti-reflection layer (n2^2 = n1 n3, a quarter wave): everything goes through
    n3 = 1.2
    nf = math.sqrt(1.69 * n3)
    out = shoot(*film_column(n3, nf, 0.0, 175.0 / (4 * nf), 1.0), n, seed=3)
    assert int(out["chan_count"][1]) == n
    # oblique: transmitted photons obey Snell into medium 3 and arrive at the top detector; the reflected ones return to the bottom
    # (start at x = -35 mm: the reflected photon is 70 mm further in x when it is back at z = 0, the sheets reach to +-50 mm)
    out = shoot(*film_column(1.6, 0.81, 1.86, 15.0, 0.0), n, theta_deg=25.0, seed=4, x0=-35.0)
    assert int(out["fate_count"][orc.FATE_ESCAPED]) == 0
    Rs, _, Ts, _ = orc.film_coefficients(1.69, 0.81, 1.86, 15.0, 1.6, 175.0, math.cos(math.radians(25.0)))
    c = out["chan_count"].astype(float) / n
    assert abs(c[0] - Rs) < sig(Rs) and abs(c[1] - Ts) < sig(Ts) and c[2] == 0
    top = out["channel"] == 1
    sin3 = np.hypot(out["dir"][0][top], out["dir"][1][top])
    assert np.abs(1.6 * sin3 - 1.69 * math.sin(math.radians(25.0))).max() < 1e-6
