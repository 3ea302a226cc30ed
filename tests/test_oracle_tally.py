"""Pins of the design-study reductions: they are defined as counting."""
import math

import numpy as np

from oracle import oracle as orc


def test_tally_on_a_hand_made_case():
    D, B, S, E = orc.FATE_DETECTED, orc.FATE_BULK_ABSORBED, orc.FATE_SURFACE_ABSORBED, orc.FATE_ESCAPED
    #           source 0                 | source 1                  | source 2 (ragged: one photon)
    fate = [D, D, B, S,                    S, S, D, E,                 D]
    chan = [0, 3, -1, -1,                  -1, -1, 2, -1,              7]            # channel 7 does not exist: not counted in any group
    t = [0.5, 2.2, 9.0, 9.0,               1.0, 1.0, 99.0, 0.0,        -3.0]
    last = [10, 11, -1, 4,                 5, 99, 12, -1,              13]           # triangle 99 does not exist
    flags = np.array(fate, np.uint32) | 0x40                                          # history bits must not matter
    group = np.array([0, 0, 1, 1], np.int32)                                          # channels 0,1 bottom; 2,3 top
    comp = np.full(20, 2, np.int32); comp[4] = 0; comp[5] = 1
    r = orc.tally(flags, np.array(chan), np.array(t, np.float32), np.array(last), 4, group, 2, comp, 3, n_bins=4, t_min=0.0, dt=1.0)
    assert r["detected"].tolist() == [[1, 1], [0, 1], [0, 0]]
    assert r["time_hist"].tolist() == [[1, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0]]      # 99 ns -> last bin, -3 ns -> first bin
    assert r["fate_by_source"][:, :4].tolist() == [[2, 1, 1, 0], [1, 0, 2, 1], [1, 0, 0, 0]]
    assert r["absorbed_by_component"].tolist() == [1, 1, 0]                           # the hit on triangle 99 is not attributed
    assert int(r["fate_by_source"].sum()) == 9


def test_t90_definition():
    rng = np.random.default_rng(1)
    tau, n = 27.0, 2_000_000
    t = rng.exponential(tau, n)
    h, _ = np.histogram(t, bins=4000, range=(0.0, 400.0))
    t90 = orc.t90_from_hist(h, 0.0, 0.1)
    assert abs(t90 - tau * math.log(10.0)) < 0.15                                     # closed form for an exponential: tau ln 10 = 62.17 ns
    assert abs(t90 - np.quantile(t, 0.9)) < 0.1                                        # and the plain quantile of the same sample
    assert orc.t90_from_hist([0, 10, 0, 0], 5.0, 2.0) == 5.0 + 2.0 * (1 + 0.9)         # all in one bin: linear inside it
    assert math.isnan(orc.t90_from_hist([0, 0], 0.0, 1.0))
    assert abs(orc.t90_from_hist(h, 0.0, 0.1, q=0.5) - tau * math.log(2.0)) < 0.1
