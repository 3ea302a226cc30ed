"""Pins of the oracle's emission: closed-form laws the paper and the mathematics fix.

PAPER.md line 144: Gaussian spectrum, mean 174.8 nm, FWHM 10.2 nm; two-component exponential time profile.
Table 2 (lines 155-160): tau_1 = 3.5 ns, tau_3 = 24 ns, f_s = 0.66 (NR) / 0.22 (ER).  Line 191: isotropic, uniform in the volume.
"""
import math

import numpy as np
from scipy import stats

from oracle import oracle as orc
from paper_2203_14354_b200 import synth

N = 400_000
P_MIN = 1e-4        # one-sample KS at fixed seeds; a wrong law fails by many orders of magnitude


def ks_uniform(x):
    return stats.kstest(x, "uniform").pvalue


def test_cylinder_positions_are_uniform_in_the_volume():
    src = synth.source(synth.SHAPE_CYLINDER, (10.0, -20.0, 0.0), 1299.0, 2.0, 2599.0)
    r = orc.emit(src, 11, 0, N)
    dx, dy, z = r["pos"][0] - 10.0, r["pos"][1] + 20.0, r["pos"][2]
    rho2 = (dx * dx + dy * dy) / 1299.0 ** 2
    assert rho2.max() <= 1.0 and z.min() >= 2.0 and z.max() <= 2599.0
    assert ks_uniform(rho2) > P_MIN                                   # area element r dr: r^2 uniform
    assert ks_uniform((np.arctan2(dy, dx) + math.pi) / (2 * math.pi)) > P_MIN
    assert ks_uniform((z - 2.0) / 2597.0) > P_MIN
    assert abs(z.mean() - 1300.5) < 5 * 2597.0 / math.sqrt(12 * N)
    # r^2, azimuth and z are independent: correlations vanish
    for a, b in ((rho2, z), (rho2, np.arctan2(dy, dx)), (z, np.arctan2(dy, dx))):
        assert abs(np.corrcoef(a, b)[0, 1]) < 5 / math.sqrt(N)


def test_ball_and_point_positions():
    src = synth.source(synth.SHAPE_BALL, (400.0, 200.0, 2601.25), 1.0)
    r = orc.emit(src, 12, 0, N)
    d = r["pos"] - np.array([[400.0], [200.0], [2601.25]])
    rho = np.sqrt((d * d).sum(0))
    assert rho.max() <= 1.0 + 1e-12
    assert ks_uniform(rho ** 3) > P_MIN                               # volume element rho^2 d rho
    assert ks_uniform((d[2] / rho + 1) / 2) > P_MIN                   # direction of the offset is isotropic
    assert np.abs(d.mean(1)).max() < 5 * math.sqrt(0.2 / N)           # <x^2> = R^2 / 5 per axis
    p = orc.emit(synth.source(synth.SHAPE_POINT, (1.5, -2.5, 3.5)), 13, 0, 1000)
    assert np.all(p["pos"] == np.array([[1.5], [-2.5], [3.5]]))


def test_directions_isotropic_and_polarisation_random_transverse():
    r = orc.emit(synth.source_for(2), 14, 0, N)
    k, e = r["dir"], r["pol"]
    assert np.abs((k * k).sum(0) - 1).max() < 1e-12 and np.abs((e * e).sum(0) - 1).max() < 1e-12
    assert np.abs((k * e).sum(0)).max() < 1e-12                       # transverse
    assert ks_uniform((k[2] + 1) / 2) > P_MIN                         # cos(theta) uniform
    assert ks_uniform((np.arctan2(k[1], k[0]) + math.pi) / (2 * math.pi)) > P_MIN
    assert np.abs(k.mean(1)).max() < 5 * math.sqrt(1 / (3 * N))
    # azimuth of e about k, measured in any frame that depends on k only, is uniform
    ref = np.where(np.abs(k[0]) < 0.5, 1.0, 0.0)[None, :] * np.array([[1.0], [0.0], [0.0]]) + \
          np.where(np.abs(k[0]) < 0.5, 0.0, 1.0)[None, :] * np.array([[0.0], [1.0], [0.0]])
    a = np.cross(ref.T, k.T).T
    a /= np.sqrt((a * a).sum(0))
    b = np.cross(k.T, a.T).T
    psi = np.arctan2((e * b).sum(0), (e * a).sum(0))
    assert ks_uniform((psi + math.pi) / (2 * math.pi)) > P_MIN
    # and e itself is isotropic over the sphere (second moments 1/3, no preferred axis)
    assert np.abs((e * e).mean(1) - 1 / 3).max() < 5 * math.sqrt(4 / 45 / N)


def test_spectrum_is_the_papers_gaussian():
    r = orc.emit(synth.source_for(2), 15, 0, N)
    lam = r["wavelength"]
    sigma = 10.2 / (2 * math.sqrt(2 * math.log(2)))
    assert stats.kstest(lam, stats.norm(174.8, sigma).cdf).pvalue > P_MIN
    assert abs(lam.mean() - 174.8) < 5 * sigma / math.sqrt(N)
    # the definition of FWHM: the density at mean +- FWHM/2 is half the peak, so P(|lambda - mean| < FWHM/2) = erf(sqrt(ln 2))
    inside = (np.abs(lam - 174.8) < 5.1).mean()
    p = math.erf(math.sqrt(math.log(2)))
    assert abs(p - 0.7610) < 1e-3 and abs(inside - p) < 5 * math.sqrt(p * (1 - p) / N)
    mono = orc.emit(synth.source(synth.SHAPE_POINT, lambda_mean=175.0, lambda_fwhm=0.0), 15, 0, 100)
    assert np.all(mono["wavelength"] == 175.0)


def test_time_profile_is_two_exponentials():
    for fs, seed in ((0.66, 16), (0.22, 17)):
        src = synth.source(synth.SHAPE_POINT, f_singlet=fs, t_start=5.0)
        t = orc.emit(src, seed, 0, N)["t0"] - 5.0
        assert t.min() > 0
        cdf = lambda x: fs * (1 - np.exp(-x / 3.5)) + (1 - fs) * (1 - np.exp(-x / 24.0))
        assert stats.kstest(t, cdf).pvalue > P_MIN
        mean = fs * 3.5 + (1 - fs) * 24.0
        var = fs * 2 * 3.5 ** 2 + (1 - fs) * 2 * 24.0 ** 2 - mean ** 2
        assert abs(t.mean() - mean) < 5 * math.sqrt(var / N)
    one = orc.emit(synth.source(synth.SHAPE_POINT, tau1=27.0, tau3=27.0, f_singlet=1.0), 18, 0, N)["t0"]
    assert stats.kstest(one, stats.expon(0, 27.0).cdf).pvalue > P_MIN   # BASELINE.json configs[4]: exp(tau = 27 ns)


def test_emission_is_a_function_of_seed_and_photon_id_only():
    src = synth.source_for(2)
    whole = orc.emit(src, 21, 1000, 5000)
    part = orc.emit(src, 21, 3000, 1000)
    for key in ("pos", "dir", "pol", "wavelength", "t0"):
        assert np.array_equal(whole[key][..., 2000:3000], part[key])
    other = orc.emit(src, 22, 1000, 5000)
    assert not np.array_equal(whole["wavelength"], other["wavelength"])
    # a two-source batch (dw_emit_sources: photon i belongs to source i // m, ids base + i) is the two single-source batches one
    # after the other: nothing of a photon depends on its neighbours or on where its batch starts
    a, b, m = synth.source_for(4), synth.source(synth.SHAPE_POINT, (1.0, 2.0, 3.0)), 700
    ids = np.arange(9000, 9000 + 2 * m)
    for s_, one in ((a, slice(0, m)), (b, slice(m, 2 * m))):
        full = orc.emit(s_, 21, 9000, 2 * m)
        alone = orc.emit(s_, 21, int(ids[one][0]), m)
        for key in ("pos", "dir", "pol", "wavelength", "t0"):
            assert np.array_equal(full[key][..., one], alone[key])
    # the draws are the documented Philox blocks of step 0xFFFFFFFF (guards the counter layout, not the laws)
    u = orc.uniforms(21, 1000, 0xFFFFFFFF, 0)
    assert abs(whole["pos"][2][0] - (2.0 + 2597.0 * u[2])) < 1e-9
