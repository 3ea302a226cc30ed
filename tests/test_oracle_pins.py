"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each check compares the oracle with something other than
itself: values printed in the paper (tests/golden/), closed forms written in a different algebraic form
than the oracle's code, linear-algebra definitions, or published known-answer vectors.
"""
import math

import numpy as np
import pytest
from scipy import stats

from oracle import oracle as orc
from paper_2203_14354_b200 import synth

N_LXE, N_GXE, N_QUARTZ = 1.69, 1.0, 1.60   # Table 2


def optics_custom(n, la, ls, det, rd, rs, tr):
    f = lambda v: np.asarray(v, np.float32)[:, None].copy()
    return synth.Optics(1, 175.0, 1.0, f(n), f(la), f(ls), f(det), f(rd), f(rs), f(tr))


def fates(out):
    return {name: int(out["fate_count"][i]) for i, name in enumerate(orc.FATE_NAMES)}


def photons_from(pos, k, e, t0=None):
    pos, k, e = (np.ascontiguousarray(np.asarray(a, np.float32)) for a in (pos, k, e))
    n = pos.shape[1]
    return synth.Photons(pos, k, e, np.full(n, 175.0, np.float32),
                         np.zeros(n, np.float32) if t0 is None else np.asarray(t0, np.float32))


# ----------------------------------------------------------------------------- S12 RNG
def test_philox_known_answers(golden):
    rows = golden("philox4x32_10_kat.txt")
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert list(orc.philox4x32_10(v[0:4], v[4:6])) == v[6:10]


def test_uniform_mapping_open_interval_and_fp32_exact():
    u = np.array([orc.uniforms(7, p, s, b) for p in range(50) for s in range(3) for b in range(2)])
    assert u.min() > 0 and u.max() < 1
    assert np.all(u.astype(np.float32).astype(np.float64) == u)      # exactly representable in fp32
    assert np.all((u * 2 ** 23 - 0.5) == np.round(u * 2 ** 23 - 0.5))  # ((x>>9)+0.5) 2^-23
    # distinct (photon, step, block) -> distinct streams
    assert len({tuple(r) for r in u}) == len(u)
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / u.size)


# ----------------------------------------------------------------------------- P1 first hit
def test_first_hit_from_centre_is_cone_membership():
    """A ray from the origin hits triangle T iff its direction is a non-negative combination of T's
    vertices (linear-algebra definition, np.linalg.solve), at d = 1 / sum(w)."""
    g = synth.sphere_detector(1000.0, 2)   # 320 triangles
    o = orc.Oracle(g, synth.default_optics(), bvh=False)
    rng = np.random.default_rng(0)
    k = synth.isotropic(rng, 300)
    tri, d = o.first_hit(np.zeros((3, 300)), k)
    k32 = k.astype(np.float32).astype(np.float64)
    V = g.xyz.astype(np.float64)
    for i in range(300):
        M = V[g.idx[tri[i]]].T                      # columns v0 v1 v2
        w = np.linalg.solve(M, k32[:, i])
        assert np.all(w > -1e-12), (i, w)
        assert d[i] == pytest.approx(1.0 / w.sum(), rel=1e-12)
        others = [t for t in range(g.n_tri) if t != tri[i]]
        W = np.linalg.solve(V[g.idx[others]].transpose(0, 2, 1), np.broadcast_to(k32[:, i], (len(others), 3))[..., None])[..., 0]
        assert not np.any(np.all(W > 1e-12, axis=1))  # no other triangle strictly contains the ray


def test_first_hit_icosphere_analytic_bound():
    g = synth.sphere_detector(1000.0, 4)
    o = orc.Oracle(g, synth.default_optics(), bvh=True)
    k = synth.isotropic(np.random.default_rng(1), 20000)
    tri, d = o.first_hit(np.zeros((3, 20000)), k)
    assert np.all(tri >= 0)
    V = g.xyz.astype(np.float64)
    p0, p1, p2 = (V[g.idx[:, j]] for j in range(3))
    nrm = np.cross(p1 - p0, p2 - p0)
    nrm /= np.linalg.norm(nrm, axis=1)[:, None]
    inradius = np.einsum("ij,ij->i", nrm, p0).min()     # nearest facet plane
    assert inradius > 1000.0 * 0.998
    assert d.min() >= inradius - 1e-9 and d.max() <= 1000.0 + 1e-3   # fp32 vertices sit on R to 1e-4


def test_first_hit_cube_faces_and_seam_tiebreak():
    g = synth.box((-1, -2, -3), (1, 2, 3), 0, 2, 0)
    o = orc.Oracle(g, synth.default_optics(), bvh=False)
    rng = np.random.default_rng(2)
    k = synth.isotropic(rng, 2000).astype(np.float32)
    tri, d = o.first_hit(np.zeros((3, 2000)), k)
    h = np.array([1.0, 2.0, 3.0])
    expect = (h[:, None] / np.abs(k.astype(np.float64))).min(axis=0)   # slab exit distance of a box
    assert np.allclose(d, expect, rtol=1e-12)
    # seam (appendix item 2): a ray aimed exactly at the diagonal shared by the two
    # triangles of the +z face is hit exactly once, by the lower id; never dropped.
    tri2, d2 = o.first_hit(np.zeros((3, 1)), np.array([[0.0], [0.0], [1.0]]))
    assert d2[0] == 3.0 and tri2[0] == 2      # triangles 2,3 form the +z face (synth.box order)
    # a ray aimed exactly at a cube corner / edge is still a hit
    tri3, d3 = o.first_hit(np.zeros((3, 2)), np.array([[1.0, 1.0], [2.0, 0.0], [3.0, 3.0]]) / np.array([math.sqrt(14), math.sqrt(10)]))
    assert np.all(tri3 >= 0)
    # exclusion removes the nearest triangle and exposes the co-located neighbour
    tri4, d4 = o.first_hit(np.zeros((3, 1)), np.array([[0.0], [0.0], [1.0]]), exclude=np.array([2], np.int32))
    assert tri4[0] == 3 and d4[0] == 3.0


@pytest.mark.parametrize("cfg", [0, 1])
def test_own_bvh_equals_brute_force(cfg):
    c = synth.config(cfg)
    o = orc.Oracle(c.geometry, c.optics, bvh=True)
    n = 4000
    ph = c.make_photons(n)
    tb, db = o.first_hit(ph.pos, ph.dir, use_bvh=False)
    tv, dv = o.first_hit(ph.pos, ph.dir, use_bvh=True)
    assert np.array_equal(tb, tv) and np.array_equal(db, dv)
    # second set: origins on surfaces, previous triangle excluded, new random directions
    x = ph.pos.astype(np.float64) + db * ph.dir.astype(np.float64)
    k2 = synth.isotropic(np.random.default_rng(5), n)
    tb2, db2 = o.first_hit(x, k2, exclude=tb, use_bvh=False)
    tv2, dv2 = o.first_hit(x, k2, exclude=tb, use_bvh=True)
    assert np.array_equal(tb2, tv2) and np.array_equal(db2, dv2)
    assert not np.any(tb2 == tb)


# ----------------------------------------------------------------------------- P2 absorption
def test_absorbing_sphere_exp_minus_half():
    """BASELINE.json configs[0]: detected fraction exp(-R/L_abs) = exp(-0.5)."""
    c = synth.config(0)
    o = orc.Oracle(c.geometry, c.optics, bvh=True)
    ph = c.make_photons(c.n_photons)
    out = o.propagate(ph, c.seed, c.max_steps)
    f = fates(out)
    N = c.n_photons
    p = math.exp(-0.5)
    sigma = math.sqrt(p * (1 - p) / N)
    assert abs(f["detected"] / N - p) < 4 * sigma + 2e-4     # +2e-4: faceting (d slightly < R)
    assert f["detected"] + f["bulk_absorbed"] == N
    assert f["escaped"] == f["truncated"] == f["nan_abort"] == f["surface_absorbed"] == 0
    assert int(out["total_steps"][0]) == N and np.all(out["steps"] == 1)
    assert int(out["chan_count"].sum()) == f["detected"]
    # detected photons sit on the mesh, absorbed ones inside; time = path / c with n = 1
    r = np.linalg.norm(out["pos"], axis=0)
    det = out["fate"] == orc.FATE_DETECTED
    assert np.all(r[det] > 997.0) and np.all(r[~det] < 1000.0)
    assert np.allclose(out["t"], r / 299.792458, rtol=1e-6)   # fp32 input directions: |k| = 1 +- 1e-7
    # absorbed path lengths are exponential with mean L truncated at R: KS against the closed form
    L = 2000.0
    cdf = lambda x: (1 - np.exp(-x / L)) / (1 - math.exp(-997.0 / L))
    sel = (~det) & (r < 997.0)
    assert stats.kstest(r[sel], cdf).pvalue > 1e-3


def test_bulk_competition_closed_forms():
    """P2b: with absorption and scattering both on, first event is an absorption with probability
    (1/La)/(1/La+1/Ls); unscattered-detected fraction from the centre is exp(-R(1/La+1/Ls))."""
    g = synth.sphere_detector(1000.0, 3)
    La, Ls = 1500.0, 700.0
    op = optics_custom([1.3] * 4, [La] * 4, [Ls] * 4, [0, 0, 0, 1], [0] * 4, [0] * 4, [0] * 4)
    o = orc.Oracle(g, op, bvh=True)
    N = 200_000
    ph = synth.photons_point(11, N)
    one = o.propagate(ph, 11, 1)
    fate = one["fate"]
    absorbed = (fate == orc.FATE_BULK_ABSORBED).sum()
    scattered = ((fate == orc.FATE_TRUNCATED) & ((one["flags"] & orc.H_RAYLEIGH) != 0)).sum()
    p = (1 / La) / (1 / La + 1 / Ls)
    nb = absorbed + scattered
    assert abs(absorbed / nb - p) < 4 * math.sqrt(p * (1 - p) / nb)
    # distance to the first bulk event is exponential with rate 1/La + 1/Ls (truncated at the wall)
    r = np.linalg.norm(one["pos"], axis=0)[fate != orc.FATE_DETECTED]
    lam = 1 / La + 1 / Ls
    assert stats.kstest(r[r < 990], lambda x: (1 - np.exp(-lam * x)) / (1 - math.exp(-lam * 990))).pvalue > 1e-3
    full = o.propagate(ph, 11, 1000)
    unsc = ((full["fate"] == orc.FATE_DETECTED) & ((full["flags"] & orc.H_RAYLEIGH) == 0)).sum()
    q = math.exp(-1000.0 * lam)
    assert abs(unsc / N - q) < 4 * math.sqrt(q * (1 - q) / N) + 2e-4
    assert int(full["fate_count"].sum()) == N


def test_time_of_flight_uses_refractive_index():
    """S5: crossing 2600 mm of LXe (n = 1.69) takes 14.66 ns (paper's t90 >> this)."""
    g = synth.box((-10, -10, 0), (10, 10, 2600), 0, 2, 3)
    op = synth.default_optics()
    op.abs_len[:] = np.inf
    op.scat_len[:] = np.inf
    o = orc.Oracle(g, op, bvh=False)
    ph = photons_from([[0], [0], [0.0]], [[0], [0], [1]], [[1], [0], [0]])
    ph.pos[2, 0] = 1e-3
    out = o.propagate(ph, 1, 5)
    assert out["fate"][0] == orc.FATE_DETECTED
    assert out["t"][0] == pytest.approx((2600 - 1e-3) * 1.69 / 299.792458, rel=1e-7)
    assert out["t"][0] == pytest.approx(14.66, abs=0.01)


# ----------------------------------------------------------------------------- P3 / P4 Fresnel
def _fresnel_sine_forms(n1, n2, ti):
    """Textbook Fresnel in sine/tangent form (different algebra from the oracle's amplitude ratios)."""
    tt = math.asin(n1 / n2 * math.sin(ti))
    Rs = (math.sin(ti - tt) / math.sin(ti + tt)) ** 2
    Rp = (math.tan(ti - tt) / math.tan(ti + tt)) ** 2
    return Rs, Rp, tt


def _incidence(theta, pol_angle=0.0):
    """k in the x-z plane hitting a surface whose facing normal is +z... photon travels towards -z."""
    k = np.array([math.sin(theta), 0.0, -math.cos(theta)])
    s = np.array([0.0, 1.0, 0.0])
    p = np.cross(s, k)
    e = math.cos(pol_angle) * s + math.sin(pol_angle) * p
    return k, e, np.array([0.0, 0.0, 1.0])


def test_fresnel_coefficients_against_sine_tangent_forms():
    for n1, n2 in ((N_LXE, N_GXE), (N_GXE, N_LXE), (N_GXE, N_QUARTZ), (N_LXE, N_QUARTZ)):
        for deg in (1.0, 10.0, 20.0, 30.0, 35.0):
            ti = math.radians(deg)
            Rs, Rp, tt = _fresnel_sine_forms(n1, n2, ti)
            k, e, nh = _incidence(ti, 0.0)
            assert orc.fresnel(n1, n2, nh, k, e, 0.5)[1] == pytest.approx(Rs, rel=1e-10)
            k, e, nh = _incidence(ti, math.pi / 2)
            assert orc.fresnel(n1, n2, nh, k, e, 0.5)[1] == pytest.approx(Rp, rel=1e-9, abs=1e-15)
            k, e, nh = _incidence(ti, 0.7)
            R = orc.fresnel(n1, n2, nh, k, e, 0.5)[1]
            assert R == pytest.approx(math.cos(0.7) ** 2 * Rs + math.sin(0.7) ** 2 * Rp, rel=1e-9)
    # the two numbers quoted in SURVEY 8c P4
    Rs, Rp, _ = _fresnel_sine_forms(N_LXE, N_GXE, math.radians(20))
    assert Rs == pytest.approx(0.103131, abs=1e-6) and Rp == pytest.approx(0.035908, abs=1e-6)


def test_fresnel_normal_incidence_never_aborts_and_matches_paper(golden):
    g = {r[0]: (float(r[1]), float(r[2])) for r in golden("paper_fresnel_checks.txt")}
    k, e, nh = np.array([0, 0, -1.0]), np.array([0.6, 0.8, 0.0]), np.array([0, 0, 1.0])
    oc, R, k2, e2 = orc.fresnel(N_LXE, N_GXE, nh, k, e, 0.999)
    assert R == pytest.approx(((N_LXE - N_GXE) / (N_LXE + N_GXE)) ** 2, rel=1e-12)
    assert abs(R - g["reflect_lxe_gxe"][0]) <= g["reflect_lxe_gxe"][1] + 1e-3   # paper prints 6.5%: 0.0658
    assert oc == 1 and np.allclose(k2, k) and np.allclose(np.abs(e2 @ e), 1.0)
    oc, R, k2, e2 = orc.fresnel(N_LXE, N_GXE, nh, k, e, 0.0)
    assert oc == 0 and np.allclose(k2, -k) and np.all(np.isfinite(e2)) and abs(np.linalg.norm(e2) - 1) < 1e-12


def test_snell_brewster_critical_angles():
    # Snell + geometry of the refracted ray and polarisation
    for n1, n2, deg, psi in ((N_LXE, N_GXE, 25.0, 0.3), (N_GXE, N_QUARTZ, 60.0, 1.1), (N_LXE, N_QUARTZ, 50.0, 0.0)):
        ti = math.radians(deg)
        k, e, nh = _incidence(ti, psi)
        oc, R, k2, e2 = orc.fresnel(n1, n2, nh, k, e, 0.99999)
        assert oc == 1
        tt = math.asin(n1 / n2 * math.sin(ti))
        assert np.allclose(k2, [math.sin(tt), 0, -math.cos(tt)], atol=1e-12)
        assert abs(np.linalg.norm(e2) - 1) < 1e-12 and abs(e2 @ k2) < 1e-12
        # amplitude ratio t_p/t_s = 1/cos(ti - tt) (sine-form identity)
        s = np.array([0, 1.0, 0])
        p2 = np.cross(s, k2)
        if psi != 0.0:
            assert (e2 @ p2) / (e2 @ s) == pytest.approx(math.tan(psi) / math.cos(ti - tt), rel=1e-9)
        # reflection: angle in = angle out
        oc, R, k3, e3 = orc.fresnel(n1, n2, nh, k, e, 0.0)
        assert oc == 0 and np.allclose(k3, [math.sin(ti), 0, math.cos(ti)], atol=1e-12) and abs(e3 @ k3) < 1e-12
    # Brewster: R_p = 0 at atan(n2/n1) = 30.613 deg for LXe -> GXe
    tb = math.atan(N_GXE / N_LXE)
    assert math.degrees(tb) == pytest.approx(30.613, abs=1e-3)
    k, e, nh = _incidence(tb, math.pi / 2)
    assert orc.fresnel(N_LXE, N_GXE, nh, k, e, 0.5)[1] < 1e-20
    # critical angles 36.279 deg (LXe->GXe), 71.217 deg (LXe->quartz): R = 1 above, < 1 below
    for n2, crit in ((N_GXE, 36.279), (N_QUARTZ, 71.217)):
        assert math.degrees(math.asin(n2 / N_LXE)) == pytest.approx(crit, abs=1e-3)
        for psi in (0.0, 0.8, math.pi / 2):
            k, e, nh = _incidence(math.radians(crit + 0.01), psi)
            oc, R, k2, e2 = orc.fresnel(N_LXE, n2, nh, k, e, 0.999999)
            assert oc == 2 and R == 1.0 and k2[2] > 0 and abs(e2 @ k2) < 1e-12 and abs(np.linalg.norm(e2) - 1) < 1e-12
            k, e, nh = _incidence(math.radians(crit - 0.01), psi)
            oc, R, _, _ = orc.fresnel(N_LXE, n2, nh, k, e, 0.999999)
            assert oc == 1 and R < 1.0


def _slab_stack(bottom_window: bool):
    """Closed column: bottom PMT (ch 0) at z=0 [optionally behind an LXe/quartz window at z=5], liquid
    surface at z=100, GXe gap, quartz window at z=110, photocathode (ch 1) at z=115 inside the quartz."""
    LXE, GXE, SOLID, QUARTZ = 0, 1, 2, 3
    A = -50.0, 50.0
    def sheet(z, mi, mo, surf, ch):
        xyz = np.array([[A[0], A[0], z], [A[1], A[0], z], [A[1], A[1], z], [A[0], A[1], z]])
        return synth.Geometry(xyz.astype(np.float32), np.array([[0, 1, 2], [0, 2, 3]], np.int32),
                              np.full(2, mi, np.int32), np.full(2, mo, np.int32), np.full(2, surf, np.int32),
                              np.full(2, ch, np.int32), max(ch + 1, 0))
    parts = [sheet(0.0, QUARTZ if bottom_window else LXE, SOLID, 1, 0)]   # normal +z: inner is BELOW... see below
    # sheet() normals point +z, i.e. from inner (below) to outer (above)
    parts = [sheet(0.0, SOLID, QUARTZ if bottom_window else LXE, 1, 0)]
    if bottom_window:
        parts.append(sheet(5.0, QUARTZ, LXE, -1, -1))
    parts += [sheet(100.0, LXE, GXE, -1, -1), sheet(110.0, GXE, QUARTZ, -1, -1), sheet(115.0, QUARTZ, SOLID, 1, 1)]
    g = synth.merge(*parts)
    g.n_channels = 2
    inf = np.inf
    op = optics_custom([N_LXE, N_GXE, 1.0, N_QUARTZ], [inf] * 4, [inf] * 4, [0, 1.0], [0, 0], [0, 0], [0, 0])
    return g, op


def _slab_expectation(bottom_window: bool):
    """Absorbing Markov chain over (interface, direction) solved with numpy; normal-incidence
    reflectances from the textbook ((n1-n2)/(n1+n2))^2."""
    r = lambda a, b: ((a - b) / (a + b)) ** 2
    R1, R2, R0 = r(N_LXE, N_GXE), r(N_GXE, N_QUARTZ), (r(N_LXE, N_QUARTZ) if bottom_window else 0.0)
    # unknowns: probability of ending at the BOTTOM for a photon  a) going up in liquid (U),
    # b) going down in liquid (D), c) going up in gas (G), d) going down in gas (H)
    # U = R1*D + (1-R1)*G ; D = (1-R0)*1 + R0*U ; G = R2*H + (1-R2)*0 ; H = (1-R1)*D + R1*G
    A = np.array([[1, -R1, -(1 - R1), 0], [-R0, 1, 0, 0], [0, 0, 1, -R2], [0, -(1 - R1), -R1, 1]], float)
    b = np.array([0, 1 - R0, 0, 0], float)
    U = np.linalg.solve(A, b)[0]
    return U, R1, (1 - R1) * R2 * (1 - R1)


@pytest.mark.parametrize("bottom_window", [False, True])
def test_paper_normal_incidence_check(golden, bottom_window):
    """photons straight up from the liquid: 6.5% reflect at LXe/GXe, 4.6% (of all)
    reflect at GXe/quartz and return, 11.2% bottom / 88.8% top."""
    gold = {r[0]: (float(r[1]), float(r[2])) for r in golden("paper_fresnel_checks.txt")}
    g, op = _slab_stack(bottom_window)
    o = orc.Oracle(g, op, bvh=False)
    N = 400_000
    rng = np.random.default_rng(3)
    pos = np.stack([rng.uniform(-40, 40, N), rng.uniform(-40, 40, N), np.full(N, 50.0)])
    k = np.zeros((3, N)); k[2] = 1
    psi = rng.uniform(0, 2 * np.pi, N)
    e = np.stack([np.cos(psi), np.sin(psi), np.zeros(N)])
    out = o.propagate(photons_from(pos, k, e), 5, 100)
    f = fates(out)
    assert f["detected"] == N
    bottom = int(out["chan_count"][0]) / N
    top = int(out["chan_count"][1]) / N
    U, R1, T1R2T1 = _slab_expectation(bottom_window)
    sig = math.sqrt(U * (1 - U) / N)
    assert abs(bottom - U) < 4 * sig and abs(top - (1 - U)) < 4 * sig
    assert U == pytest.approx(0.11236 if bottom_window else 0.11244, abs=2e-5)
    # the printed (rounded) values of the paper
    assert abs(bottom - gold["bottom_fraction"][0]) < gold["bottom_fraction"][1] + 4 * sig
    assert abs(top - gold["top_fraction"][0]) < gold["top_fraction"][1] + 4 * sig
    assert abs(R1 - gold["reflect_lxe_gxe"][0]) < 1e-3 and abs(T1R2T1 - gold["reflect_quartz_and_return"][0]) < 1e-3
    # first-step statistics: reflected at the liquid surface on the first step
    one = o.propagate(photons_from(pos, k, e), 5, 1)
    refl = ((one["flags"] & orc.H_FRESNEL_REFLECT) != 0).mean()
    assert abs(refl - R1) < 4 * math.sqrt(R1 * (1 - R1) / N)
    assert abs(refl - gold["reflect_lxe_gxe"][0]) < gold["reflect_lxe_gxe"][1] + 4 * math.sqrt(R1 / N) + 3e-4


def test_paper_total_internal_reflection_at_75_degrees(golden):
    """100% of photons at 75 deg on the LXe/quartz window are reflected."""
    g, op = _slab_stack(True)
    o = orc.Oracle(g, op, bvh=False)
    N = 20000
    rng = np.random.default_rng(4)
    th = math.radians(75.0)
    pos = np.stack([rng.uniform(-5, 5, N), rng.uniform(-5, 5, N), np.full(N, 6.0)])
    k = np.tile(np.array([[math.sin(th)], [0.0], [-math.cos(th)]]), (1, N))
    e = synth.transverse_pol(rng, k)
    out = o.propagate(photons_from(pos, k, e), 6, 1)
    assert np.all((out["flags"] & orc.H_TIR) != 0)
    assert np.all(out["dir"][2] > 0) and np.allclose(out["dir"][2], math.cos(th), atol=1e-6)


# ----------------------------------------------------------------------------- P5 Rayleigh
def test_rayleigh_matches_theoretical_distribution():
    """PAPER.md lines 438-442 / Fig. 13: the scattering-angle distribution must be the theoretical one,
    pdf(cos theta) = 3/8 (1 + cos^2 theta) for unpolarised light; mu = e.k' has pdf 3/4 (1 - mu^2)."""
    g = synth.sphere_detector(1.0e6, 1)
    op = optics_custom([1.0] * 4, [np.inf] * 4, [1.0] * 4, [0, 0, 0, 1], [0] * 4, [0] * 4, [0] * 4)
    o = orc.Oracle(g, op, bvh=False)
    N = 300_000
    ph = synth.photons_point(21, N)
    out = o.propagate(ph, 21, 1)
    assert np.all((out["flags"] & orc.H_RAYLEIGH) != 0) and np.all(out["fate"] == orc.FATE_TRUNCATED)
    k0, e0 = ph.dir.astype(np.float64), ph.pol.astype(np.float64)
    k1, e1 = out["dir"], out["pol"]
    ct = (k0 * k1).sum(0)
    mu = (e0 * k1).sum(0)
    se = lambda v: math.sqrt(v / N)
    assert abs((ct ** 2).mean() - 0.4) < 4 * se(np.var(ct ** 2))
    assert abs((mu ** 2).mean() - 0.2) < 4 * se(np.var(mu ** 2))
    assert abs(ct.mean()) < 4 * se(0.4)
    assert stats.kstest(ct, lambda x: 0.5 + (3 * x + x ** 3) / 8).pvalue > 1e-3
    assert stats.kstest(mu, lambda x: 0.5 + 0.75 * (x - x ** 3 / 3)).pvalue > 1e-3
    # exact sampler of the same law: mu = 2 cos((acos(1-2u) + 4 pi)/3)
    u = np.random.default_rng(1).uniform(0, 1, N)
    mu_ref = 2 * np.cos((np.arccos(1 - 2 * u) + 4 * np.pi) / 3)
    assert stats.ks_2samp(mu, mu_ref).pvalue > 1e-3
    # azimuth of k' about e is uniform
    a = np.cross(e0.T, k0.T).T
    phi = np.arctan2((k1 * a).sum(0), (k1 * k0).sum(0))
    assert stats.kstest((phi + np.pi) / (2 * np.pi), "uniform").pvalue > 1e-3
    # geometry of the new polarisation: unit, transverse, coplanar with e and k', same hemisphere as e
    assert np.abs(np.linalg.norm(e1, axis=0) - 1).max() < 1e-12 and np.abs((e1 * k1).sum(0)).max() < 1e-12
    assert np.abs(np.einsum("ij,ij->j", np.cross(e0.T, k1.T).T, e1)).max() < 1e-9
    assert np.all((e1 * e0).sum(0) > 0)
    # the outcome does not depend on the old direction (only on e): same e, different k -> same k'
    k_a, e_a, it_a = orc.rayleigh([0, 0, 1.0], [1.0, 0, 0], 9, 77)
    k_b, e_b, it_b = orc.rayleigh([0, 1.0, 0], [1.0, 0, 0], 9, 77)
    assert np.array_equal(k_a, k_b) and np.array_equal(e_a, e_b)
    # acceptance rate 2/3 -> mean number of iterations 3/2
    its = np.array([orc.rayleigh([0, 0, 1.0], [1.0, 0, 0], 9, i)[2] for i in range(20000)])
    assert abs(its.mean() - 1.5) < 4 * math.sqrt(0.75 / its.size)


# ----------------------------------------------------------------------------- P6 / P7 surfaces
def test_lambert_cosine_law():
    nh = np.array([0.36, -0.48, 0.8])
    ks, es = zip(*(orc.lambert(nh, 3, i) for i in range(40000)))
    k, e = np.array(ks), np.array(es)
    c = k @ nh
    assert c.min() > 0                                   # never below the surface
    assert stats.kstest(c, lambda x: x ** 2).pvalue > 1e-3   # pdf 2 cos(theta)
    assert abs(c.mean() - 2 / 3) < 4 * math.sqrt((0.5 - 4 / 9) / c.size)
    a = np.cross([1.0, 0, 0], nh); a /= np.linalg.norm(a)
    b = np.cross(nh, a)
    phi = np.arctan2(k @ b, k @ a)
    assert stats.kstest((phi + np.pi) / (2 * np.pi), "uniform").pvalue > 1e-3
    assert np.abs(np.linalg.norm(k, axis=1) - 1).max() < 1e-12
    assert np.abs(np.linalg.norm(e, axis=1) - 1).max() < 1e-12 and np.abs((k * e).sum(1)).max() < 1e-12
    # polarisation direction uniform in the transverse plane: <(e.t)^2> = 1/2 for a transverse t
    t = np.cross(k, nh); t /= np.linalg.norm(t, axis=1)[:, None]
    assert abs(((e * t).sum(1) ** 2).mean() - 0.5) < 4 * math.sqrt(0.125 / c.size)


def test_specular_reflection_including_normal_incidence():
    """PAPER.md line 436 (appendix item 1): normal incidence must not abort a specular reflection."""
    nh = np.array([0, 0, 1.0])
    k, e = orc.specular(nh, [0, 0, -1.0], [1.0, 0, 0])
    assert np.allclose(k, [0, 0, 1]) and np.allclose(e, [1, 0, 0])
    rng = np.random.default_rng(8)
    for _ in range(100):
        kin = synth.isotropic(rng, 1)[:, 0]
        if kin[2] > 0:
            kin = -kin
        ein = synth.transverse_pol(rng, kin[:, None])[:, 0]
        k, e = orc.specular(nh, kin, ein)
        assert np.allclose(k, kin * [1, 1, -1], atol=1e-12) and abs(k @ e) < 1e-12 and abs(np.linalg.norm(e) - 1) < 1e-12
    # through the loop: a specular box, photon at normal incidence bounces between two faces for ever
    g = synth.box((-1, -1, -1), (1, 1, 1), 0, 2, 0)
    op = optics_custom([1.0] * 3, [np.inf] * 3, [np.inf] * 3, [0], [0], [1.0], [0])
    o = orc.Oracle(g, op, bvh=False)
    out = o.propagate(photons_from([[0.1], [0.2], [0.0]], [[0], [0], [1]], [[1], [0], [0]]), 1, 50)
    assert out["fate"][0] == orc.FATE_TRUNCATED and out["steps"][0] == 50
    assert (out["flags"][0] & orc.H_REFLECT_SPECULAR) and np.allclose(out["pos"][:2, 0], [0.1, 0.2])
    assert out["t"][0] == pytest.approx((1 + 49 * 2) / 299.792458, rel=1e-12)


def test_seam_between_two_reflecting_planes_is_not_lost():
    """PAPER.md line 437 (appendix item 2): a photon aimed at the joint of two wall panels must be
    reflected, not lost.  Wall segments 255 and 0 of the C1 wall share the vertical edge at (R, 0)."""
    c = synth.config(1)
    g = c.geometry
    o = orc.Oracle(g, c.optics, bvh=False)
    tri, d = o.first_hit(np.array([[0.0], [0.0], [250.0]]), np.array([[1.0], [0.0], [0.0]]))
    assert d[0] == 250.0
    cands = [t for t in range(g.n_tri) if np.any(np.all(g.xyz[g.idx[t]][:, :2] == [250.0, 0.0], axis=1)) and g.surface[t] == 0
             and g.xyz[g.idx[t]][:, 2].min() <= 250.0 <= g.xyz[g.idx[t]][:, 2].max()]
    hitters = [t for t in cands if o.first_hit(np.array([[0.0], [0.0], [250.0]]), np.array([[1.0], [0.0], [0.0]]),
                                               exclude=np.array([tt for tt in [tri[0]]], np.int32))[0][0] == t or t == tri[0]]
    assert tri[0] == min(hitters) and len(hitters) >= 2     # several triangles own the point; lowest id wins
    op = synth.default_optics(1.0)
    op.abs_len[:] = np.inf; op.scat_len[:] = np.inf
    o2 = orc.Oracle(g, op, bvh=False)
    out = o2.propagate(photons_from([[0.0], [0.0], [250.0]], [[1.0], [0], [0]], [[0], [1.0], [0]]), 3, 1)
    assert (out["flags"][0] & orc.H_REFLECT_DIFFUSE) and out["fate"][0] == orc.FATE_TRUNCATED
    assert out["dir"][0, 0] < 0 or abs(out["dir"][1, 0]) > 0    # sent back into the volume


def _random_detector_sphere(f_target, rho, subdiv=4, seed=0):
    g = synth.sphere_detector(1000.0, subdiv, material=1, surface=0)   # inner 1 / outer 2: no bulk process in either
    rng = np.random.default_rng(seed)
    V = g.xyz.astype(np.float64)
    area = 0.5 * np.linalg.norm(np.cross(V[g.idx[:, 1]] - V[g.idx[:, 0]], V[g.idx[:, 2]] - V[g.idx[:, 0]]), axis=1)
    det = rng.uniform(0, 1, g.n_tri) < f_target
    g.surface[det] = 1
    g.channel[:] = -1
    g.channel[det] = 0
    g.n_channels = 1
    f = area[det].sum() / area.sum()
    op = optics_custom([1.0] * 3, [np.inf] * 3, [np.inf] * 3, [0, 1.0], [rho, 0], [0, 0], [0, 0])
    return g, op, f


def test_integrating_sphere():
    """P8: Lambertian sphere of reflectivity rho with an area fraction f of perfect detectors:
    P_det = f / (1 - rho (1 - f)); mean number of reflections q/(1-q), q = rho (1 - f)."""
    rho = 0.95
    g, op, f = _random_detector_sphere(0.1, rho)
    o = orc.Oracle(g, op, bvh=True)
    N = 200_000
    out = o.propagate(synth.photons_point(31, N), 31, 5000)
    fc = fates(out)
    assert fc["detected"] + fc["surface_absorbed"] == N
    p = f / (1 - rho * (1 - f))
    assert abs(fc["detected"] / N - p) < 4 * math.sqrt(p * (1 - p) / N) + 1e-3
    q = rho * (1 - f)
    nrefl = out["steps"].astype(np.float64) - 1
    assert abs(nrefl.mean() - q / (1 - q)) < 4 * math.sqrt(q / (1 - q) ** 2 / N) + 0.03
    # mean total path = R + (4R/3) q/(1-q): Lambertian chords in a sphere average 4R/3
    path = out["t"] * 299.792458
    # (the inscribed, faceted icosphere sits 0.4-1.3% below the perfect-sphere closed forms; the deficit
    #  halves with each subdivision level: 1.27% / 0.70% / 0.36% at levels 3 / 4 / 5)
    assert path.mean() == pytest.approx(1000.0 + 4000.0 / 3 * q / (1 - q), rel=1e-2)
    assert int(out["chan_count"][0]) == fc["detected"]


# ----------------------------------------------------------------------------- S13 reductions are plain counting
def test_time_histogram_and_channel_counts_are_counts_of_the_per_photon_outputs():
    """S13 (arrival times of the detected photons; line 189: photons per sensor): orc_propagate's time_hist must be
    numpy's histogram of its own per-photon t over the detected photons, bins [t_min + k dt, t_min + (k + 1) dt), with earlier
    arrivals in the first bin and later ones in the last; chan_count must be numpy's bincount of its own per-photon channel.  The
    range (5 ns, 50 bins of 0.7 ns) is chosen so that both clamps are hit on C1."""
    c = synth.config(1)
    o = orc.Oracle(c.geometry, c.optics, bvh=True)
    N, t_min, dt, nb = 40000, 5.0, 0.7, 50
    out = o.propagate(c.make_photons(N), c.seed, c.max_steps, n_bins=nb, t_min=t_min, dt=dt, full=False)
    det = out["fate"] == orc.FATE_DETECTED
    t = out["t"][det]
    edges = t_min + dt * np.arange(nb + 1)
    want, _ = np.histogram(t, bins=edges)
    want = want.astype(np.uint64)
    below, above = int((t < edges[0]).sum()), int((t > edges[-1]).sum())
    assert below > 100 and above > 100                      # both clamps are exercised
    want[0] += below
    want[-1] += above
    assert np.array_equal(out["time_hist"], want)
    assert np.array_equal(out["chan_count"], np.bincount(out["channel"][det], minlength=o.n_chan).astype(np.uint64))
    # a one-bin histogram holds everything; no histogram asked for is no histogram
    one = o.propagate(c.make_photons(2000), c.seed, c.max_steps, n_bins=1, t_min=1e9, dt=1.0, full=False)
    assert one["time_hist"].tolist() == [int((one["fate"] == orc.FATE_DETECTED).sum())]


# ----------------------------------------------------------------------------- P9 conservation, P11 determinism
def test_conservation_and_invariants_on_small_tpc():
    c = synth.config(1)
    o = orc.Oracle(c.geometry, c.optics, bvh=True)
    N = 20000
    ph = c.make_photons(N)
    out = o.propagate(ph, c.seed, c.max_steps, n_bins=200, t_min=0.0, dt=1.0)
    fc = fates(out)
    assert sum(fc.values()) == N and fc["nan_abort"] == 0 and fc["escaped"] == 0
    assert int(out["chan_count"].sum()) == fc["detected"] == int(out["time_hist"].sum())
    assert int(out["total_steps"][0]) == int(out["steps"].sum())
    moved = (out["flags"] & 0xFF0) != 0     # k, e rewritten at least once (else: the fp32 inputs, 1 +- 1e-7)
    assert moved.mean() > 0.9
    assert np.abs(np.linalg.norm(out["dir"], axis=0) - 1)[moved].max() < 1e-12
    assert np.abs(np.linalg.norm(out["dir"], axis=0) - 1).max() < 2e-7
    assert np.abs(np.linalg.norm(out["pol"], axis=0) - 1).max() < 2e-7
    assert np.abs((out["dir"] * out["pol"]).sum(0)).max() < 2e-7
    assert np.all(out["t"] >= 0)
    det = out["fate"] == orc.FATE_DETECTED
    assert np.all(out["channel"][det] >= 0) and np.all(out["channel"][~det] == -1)
    assert np.all(c.geometry.channel[out["last_tri"][det]] == out["channel"][det])
    # everything stays inside the closed cylinder
    r = np.hypot(out["pos"][0], out["pos"][1])
    assert r.max() <= 250.0 + 1e-6 and out["pos"][2].min() >= -1e-6 and out["pos"][2].max() <= 500.0 + 1e-6
    # QE = 0.3: detected / (detected + absorbed on a photocathode) ~ 0.3
    on_pmt = (out["last_tri"] >= 0) & (c.geometry.surface[np.maximum(out["last_tri"], 0)] == 1) & \
             ((out["fate"] == orc.FATE_DETECTED) | (out["fate"] == orc.FATE_SURFACE_ABSORBED))
    n_on = int(on_pmt.sum())
    assert abs(fc["detected"] / n_on - 0.3) < 4 * math.sqrt(0.21 / n_on)
    # P11: same seed -> identical; batch split -> identical per-photon results; BVH == brute force
    again = o.propagate(ph, c.seed, c.max_steps, n_bins=200)
    assert all(np.array_equal(out[k], again[k]) for k in ("flags", "channel", "t", "steps", "chan_count", "time_hist"))
    a, b = o.propagate(ph.slice(0, 7001), c.seed, c.max_steps), o.propagate(ph.slice(7001, N), c.seed, c.max_steps)
    for key in ("flags", "channel", "t", "steps", "last_tri"):
        assert np.array_equal(np.concatenate([a[key], b[key]]), out[key])
    assert np.array_equal(a["chan_count"] + b["chan_count"], out["chan_count"])
    brute = o.propagate(ph.slice(0, 1500), c.seed, c.max_steps, use_bvh=False)
    assert np.array_equal(brute["flags"], out["flags"][:1500]) and np.array_equal(brute["t"], out["t"][:1500])
    other = o.propagate(ph, c.seed + 1, c.max_steps)
    assert not np.array_equal(other["flags"], out["flags"])


# ----------------------------------------------------------------------------- P10 transmit / wire shadow
def test_transmitting_sheet_and_wire_shadow():
    """electrodes as sheets of 95% / 97% transparency; line 119: 200 um wires at
    5 mm pitch.  A sheet of transmit = T passes T; an 8-sided prism grid shadows width/pitch."""
    # sheet: box with a QE=1 floor; a transmit sheet across it
    floor = synth.box((-10, -10, 0), (10, 10, 20), 0, 2, 1, 0)
    sheet = synth.Geometry(np.array([[-10, -10, 10], [10, -10, 10], [10, 10, 10], [-10, 10, 10]], np.float32),
                           np.array([[0, 1, 2], [0, 2, 3]], np.int32), np.zeros(2, np.int32), np.zeros(2, np.int32),
                           np.full(2, 2, np.int32), np.full(2, -1, np.int32))
    g = synth.merge(floor, sheet)
    inf = np.inf
    op = optics_custom([1.0] * 3, [inf] * 3, [inf] * 3, [0, 1.0, 0], [0] * 3, [0] * 3, [0, 0, 0.95])
    o = orc.Oracle(g, op, bvh=False)
    N = 100_000
    rng = np.random.default_rng(12)
    pos = np.stack([rng.uniform(-9, 9, N), rng.uniform(-9, 9, N), np.full(N, 15.0)])
    k = np.zeros((3, N)); k[2] = -1
    e = np.zeros((3, N)); e[0] = 1
    out = o.propagate(photons_from(pos, k, e), 2, 10)
    fc = fates(out)
    assert abs(fc["detected"] / N - 0.95) < 4 * math.sqrt(0.95 * 0.05 / N)
    assert fc["detected"] + fc["surface_absorbed"] == N
    # wires: synthetic grid of the C3 recipe on a small radius
    mb = synth._MeshBuilder()
    synth._wire_grid(mb, 10.0, 60.0, 5.0, 0.108, 20.0, 0)
    wires = mb.build()
    g2 = synth.merge(synth.box((-80, -80, 0), (80, 80, 20), 0, 2, 1, 0), wires)
    op2 = optics_custom([1.0] * 3, [inf] * 3, [inf] * 3, [0, 1.0, 0], [0] * 3, [0] * 3, [0] * 3)  # black wires
    o2 = orc.Oracle(g2, op2, bvh=True)
    pos = np.stack([rng.uniform(-25, 25, N), rng.uniform(-20, 20, N), np.full(N, 15.0)])
    out2 = o2.propagate(photons_from(pos, k, e), 2, 10)
    shadow = 2 * 0.108 * math.cos(math.pi / 8) / 5.0       # projected width of the octagonal prism / pitch
    frac = 1 - fates(out2)["detected"] / N
    assert abs(frac - shadow) < 4 * math.sqrt(shadow * (1 - shadow) / N)
    assert shadow == pytest.approx(0.04, abs=1e-3)          # the paper's 0.2 mm / 5 mm <-> 95-96% transparency


# ----------------------------------------------------------------------------- S3 tables on more than one wavelength node
def test_table_interpolation_and_clamping():
    """S3 / G13: linear interpolation on the uniform wavelength grid, clamped at both ends.  From the centre of a detector
    sphere the time of flight is exactly d n(lambda) / c (S5) and the detected fraction is exp(-d / L_abs(lambda)) (P2), so
    both tabulated quantities are pinned against numpy's own interpolation routine: nodes, points between nodes, and
    wavelengths beyond either end of the table."""
    R = 1000.0
    g = synth.sphere_detector(R, 4)
    op = synth.dispersive_optics()
    l0, dl, nl = synth.DISPERSIVE_GRID
    grid = l0 + dl * np.arange(nl)
    lams = np.array([150.0, 165.0, 166.25, 172.5, 175.0, 178.0, 185.0, 199.0])
    n_each = 40_000
    ph = synth.photons_point(5, n_each * len(lams))
    lam = np.repeat(lams, n_each).astype(np.float32)
    ph = synth.Photons(ph.pos, ph.dir, ph.pol, lam, ph.t0, ph.id_base)
    out = orc.Oracle(g, op, bvh=True).propagate(ph, 5, 10)
    det = out["fate"] == orc.FATE_DETECTED
    d = np.sqrt((out["pos"] ** 2).sum(0))
    # material 3 (the sphere's gas): n = 1 flat, L_abs = 2000 + 40 (lambda - 175), no scattering
    L_tab = op.abs_len[synth.MAT_C0GAS].astype(np.float64)
    assert L_tab[0] != L_tab[-1]
    for k, l in enumerate(lams):
        sel = slice(k * n_each, (k + 1) * n_each)
        L = np.interp(l, grid, L_tab)                      # numpy clamps outside the grid
        expect = np.exp(-d[sel][det[sel]] / L).mean() if det[sel].any() else 0.0
        frac = det[sel].mean()
        p = math.exp(-R / L)
        assert abs(frac - p) < 4 * math.sqrt(p * (1 - p) / n_each) + 3e-4, (l, frac, p)   # + faceting bias (d <= R)
        assert abs(expect - p) < 2e-3
    # the index of refraction through the time of flight: put the dispersive LXe inside the sphere
    g2 = synth.sphere_detector(R, 4, material=synth.MAT_LXE)
    out2 = orc.Oracle(g2, op, bvh=True).propagate(ph, 6, 1)
    direct = (out2["fate"] == orc.FATE_DETECTED) & ((out2["flags"] & orc.H_RAYLEIGH) == 0)
    assert direct.sum() > 1000
    d2 = np.sqrt((out2["pos"] ** 2).sum(0))
    n_expect = np.interp(lam.astype(np.float64), grid, op.refr_index[synth.MAT_LXE].astype(np.float64))
    # S5 advances by the ray parameter along k; the float32 input directions are unit vectors only to ~6e-8, so the parameter is
    # the geometric distance divided by |k|
    knorm = np.sqrt((ph.dir.astype(np.float64) ** 2).sum(0))
    n_seen = out2["t"] * 299.792458 / (d2 / knorm)
    assert np.abs(n_seen[direct] - n_expect[direct]).max() < 1e-9
    assert n_expect.min() < 1.62 and n_expect.max() > 1.76          # the ends of the table were reached (clamped beyond)
