"""Design variants of the synthetic TPC (synth.tpc_design / config_design, the paper's section 5 studies of sensor
coverage and PMT details): facts of the generator, well-formedness seen by the oracle, and the closed form
of a photon that goes straight through a PMT window onto the photocathode."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2203_14354_b200 import synth
from test_oracle_pins import photons_from

C_MM_NS = 299.792458


@pytest.mark.parametrize("variant", synth.DESIGN_VARIANTS)
def test_generator_facts(variant):
    c = synth.config_design(variant, 1)
    g = c.geometry
    n_pmt, n_side = g.info["n_pmt_per_array"], g.info["n_side"]
    assert g.n_channels == 2 * n_pmt + n_side
    assert (n_side > 0) == (variant in ("side_sensors", "both")) and g.info["detailed_pmt"] == (variant in ("detailed_pmt", "both"))
    sens = g.channel >= 0
    assert set(np.unique(g.channel[sens])) == set(range(g.n_channels))                       # every channel has triangles
    pmt = sens & (g.channel < 2 * n_pmt)
    assert np.all(g.surface[pmt] == synth.SURF_CATHODE) and np.all(np.bincount(g.channel[pmt]) == 32)
    if n_side:
        side = g.channel >= 2 * n_pmt
        assert np.all(g.surface[side] == synth.SURF_SIPM) and np.all(np.bincount(g.channel[side] - 2 * n_pmt) == 2)
        assert n_side == g.info["side_rows"] * 256 and 10_000 <= n_side <= 100_000           # 1e4-1e5 small sensors
        r = np.hypot(g.xyz[g.idx[side], 0], g.xyz[g.idx[side], 1])
        assert r.max() < 250.0 * np.cos(np.pi / 256) - 0.9 and r.min() > 248.0               # about 1 mm in front of the flat wall segments
    if g.info["detailed_pmt"]:
        q = g.mat_inner == synth.MAT_QUARTZ
        assert q.sum() == 2 * n_pmt * (32 + 32 + 64)                                         # window face, photocathode, rim
        assert np.all(g.mat_inner[pmt] == synth.MAT_QUARTZ) and np.all(g.mat_outer[pmt] == synth.MAT_SOLID)
        face = q & (g.surface == -1)
        assert face.sum() == 2 * n_pmt * 32 and set(np.unique(g.mat_outer[face])) == {synth.MAT_LXE, synth.MAT_GXE}
        assert (g.surface == synth.SURF_BLACK).sum() == 2 * n_pmt * (64 + 64)                # rim and skirt
    o = c.optics
    assert o.refr_index.shape[0] == 5 and o.detect.shape[0] == 6
    assert float(o.detect[synth.SURF_BLACK, 0]) == 0.0 and float(o.reflect_diffuse[synth.SURF_BLACK, 0]) == 0.0


@pytest.mark.parametrize("variant", synth.DESIGN_VARIANTS)
def test_variants_are_closed_and_consistent(variant):
    """No photon may leave (G3).  And the mesh must separate what it says it separates: a photon born in the liquid that reaches a
    surface in its first step must find liquid xenon on the side it comes from (the triangle's outer material if it arrives against
    the normal, the inner one otherwise).  The check over whole tracks, from every medium, is the device's MEDIUM_MISMATCH bit in
    tests/test_gpu_design.py; it found the first version of the detailed PMT ill-formed (an open 1 mm gap under the windows, whose
    back is declared solid) after the statistics of the two sides had disagreed by 0.16 % in LCE."""
    c = synth.config_design(variant, 1)
    g = c.geometry
    o = orc.Oracle(g, c.optics, bvh=True)
    n = 30_000
    ph = c.make_photons(n)
    r = o.propagate(ph, c.seed, c.max_steps)
    fate = r["flags"] & 0xF
    assert np.bincount(fate, minlength=6)[[orc.FATE_ESCAPED, orc.FATE_NAN_ABORT]].sum() == 0
    det = r["channel"][fate == orc.FATE_DETECTED]
    n_pmt = g.info["n_pmt_per_array"]
    assert det.min() >= 0 and det.max() < g.n_channels and (det < 2 * n_pmt).sum() > 100
    if g.info["n_side"]:
        assert (det >= 2 * n_pmt).sum() > 3 * (det < 2 * n_pmt).sum()         # the wall is most of the surface of this small detector
    r1 = o.propagate(ph, c.seed, 1)
    hit = r1["last_tri"] >= 0
    assert hit.sum() > n // 4
    t = r1["last_tri"][hit]
    V = g.xyz.astype(np.float64)
    nrm = np.cross(V[g.idx[t, 1]] - V[g.idx[t, 0]], V[g.idx[t, 2]] - V[g.idx[t, 0]])
    against = np.einsum("ij,ji->i", nrm, ph.dir[:, hit].astype(np.float64)) < 0
    near = np.where(against, g.mat_outer[t], g.mat_inner[t])
    assert np.all(near == synth.MAT_LXE)


def test_straight_through_a_pmt_window_closed_form():
    """Photons aimed straight down at a bottom PMT window from 100 mm above the cap.  Those that arrive unscattered meet the face at
    normal incidence: they are reflected with ((n1 - n2) / (n1 + n2))^2, n1 = 1.69 (LXe), n2 = 1.6 (quartz); the transmitted ones
    cross 5 mm of quartz (absorption length 1 m) and are detected with the quantum efficiency 0.3; a detected photon arrives at
    (94 x 1.69 + 5 x 1.6) / c: distance in each medium times its index (S5)."""
    c = synth.config_design("detailed_pmt", 1)
    o = orc.Oracle(c.geometry, c.optics, bvh=True)
    n = 400_000
    pos = np.tile(np.array([[3.0], [2.0], [100.0]]), (1, n))
    k = np.tile(np.array([[0.0], [0.0], [-1.0]]), (1, n))
    e = np.tile(np.array([[1.0], [0.0], [0.0]]), (1, n))
    # the first step alone: scattered, absorbed, or at the face (refracted / reflected)
    r1 = o.propagate(photons_from(pos, k, e), 77, 1)
    n_refl = int(((r1["flags"] & orc.H_FRESNEL_REFLECT) != 0).sum())
    n_refr = int(((r1["flags"] & orc.H_FRESNEL_REFRACT) != 0).sum())
    p_reach = np.exp(-94.0 / 400.0) * np.exp(-94.0 / 50000.0)                 # neither scattered nor absorbed over 94 mm of LXe
    assert n_refl + n_refr == pytest.approx(n * p_reach, abs=4 * np.sqrt(n * p_reach * (1 - p_reach)))
    R = ((1.69 - 1.6) / (1.69 + 1.6)) ** 2
    assert abs(n_refl - R * (n_refl + n_refr)) < 4 * np.sqrt(R * (n_refl + n_refr))
    assert np.allclose(r1["pos"][2][(r1["flags"] & orc.H_FRESNEL_REFRACT) != 0], 6.0, atol=1e-9)     # the face is at z = 1 + 5
    # the whole track: a photon that went straight through has refracted once, nothing else, and ended at its second step
    r = o.propagate(photons_from(pos, k, e), 77, 50)
    fl = r["flags"]
    fate = fl & 0xF
    other = orc.H_RAYLEIGH | orc.H_REFLECT_DIFFUSE | orc.H_REFLECT_SPECULAR | orc.H_TIR | orc.H_FRESNEL_REFLECT
    through = ((fl & other) == 0) & ((fl & orc.H_FRESNEL_REFRACT) != 0) & (r["steps"] == 2)
    assert through.sum() == n_refr                                             # same draws: the same photons as in the first step
    ended = through & np.isin(fate, [orc.FATE_DETECTED, orc.FATE_SURFACE_ABSORBED, orc.FATE_BULK_ABSORBED])
    assert ended.sum() == through.sum()
    bulk = (through & (fate == orc.FATE_BULK_ABSORBED)).sum()
    assert abs(bulk - through.sum() * (1 - np.exp(-5.0 / 1000.0))) < 5 * np.sqrt(through.sum() * 0.005)
    at_cathode = through & (fate != orc.FATE_BULK_ABSORBED)
    det = at_cathode & (fate == orc.FATE_DETECTED)
    assert abs(det.sum() - 0.3 * at_cathode.sum()) < 4 * np.sqrt(0.21 * at_cathode.sum())
    assert np.all(r["channel"][det] == r["channel"][det][0]) and 0 <= r["channel"][det][0] < c.geometry.info["n_pmt_per_array"]
    assert np.allclose(r["t"][det], (94.0 * 1.69 + 5.0 * 1.6) / C_MM_NS, rtol=0, atol=1e-5)
