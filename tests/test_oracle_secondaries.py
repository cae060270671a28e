"""Pins for the oracle's secondary photons (reading 16): a pair event deposits
E - 2 me c^2 and two back-to-back annihilation photons of me c^2 are followed from the vertex.  The paper's
Algorithm 1 has no secondaries; the pins are what physics and the mathematics fix: energy
conservation, fate counts, the primaries' histories unchanged, isotropy, the 511 keV line, and back-to-back
emission seen in a four-wall detector."""
import math

import numpy as np
import pytest
from scipy import stats as sps

import oracle
from paper_1209_5235_b200 import workloads as W
from paper_1209_5235_b200.workloads import _Builder

ME_C2 = 0.51099895


def lead_slab(half_z):
    return W.homogeneous_slab("lead", half=(200.0, 200.0, half_z), world_half=1000.0)


def src(E):
    return W.Source(W.SRC_PENCIL, (0.0, 0.0, -500.0), (0.0, 0.0, 1.0), W.E_MONO, E)


@pytest.mark.parametrize("precision", [64, 32])
def test_pair_directions_unit_back_to_back_isotropic(precision):
    n = 20000
    w1, w2 = oracle.pair_directions(5, 0, n, precision)
    eps = 1e-14 if precision == 64 else 1e-6
    assert np.all(np.abs(np.linalg.norm(w1, axis=1) - 1) < eps)
    assert np.array_equal(w2, -w1)                                    # exactly back to back
    # isotropy: cos(theta) uniform on [-1, 1], phi uniform, no preferred axis, second moments 1/3
    assert sps.kstest(w1[:, 2], sps.uniform(-1, 2).cdf).pvalue > 1e-3
    assert sps.kstest(np.arctan2(w1[:, 1], w1[:, 0]), sps.uniform(-math.pi, 2 * math.pi).cdf).pvalue > 1e-3
    assert np.all(np.abs(w1.mean(axis=0)) < 4 / math.sqrt(3 * n))
    assert np.all(np.abs((w1 ** 2).mean(axis=0) - 1 / 3) < 4 * math.sqrt(4 / 45 / n))
    # a function of (seed, id) only
    a, _ = oracle.pair_directions(5, 100, 10, precision)
    assert np.array_equal(a, w1[100:110])
    b, _ = oracle.pair_directions(6, 0, 10, precision)
    assert not np.array_equal(b, w1[:10])


@pytest.mark.parametrize("precision", [64, 32])
def test_energy_and_fate_bookkeeping_with_secondaries(precision):
    g = lead_slab(10.0)
    og = oracle.OracleGeometry(g, secondaries=1)
    n = 4000
    r = og.transport(src(6.0), 3, n, precision)
    s = r["stats"]
    assert s["n_pair"] > n // 10                                      # the case really exercises pair events
    total = r["edep"].sum() + s["e_escaped"] + s["e_stuck"]
    assert abs(total / s["e_source"] - 1) < (1e-12 if precision == 64 else 2e-6)
    assert abs(r["edep"].sum() - s["e_deposited"]) <= 1e-9 * s["e_source"]
    # every photon ends exactly once; each pair event adds two photons, none of which can pair-produce (me c^2 < 2 me c^2)
    assert s["n_pe"] + s["n_pair"] + s["n_cut"] + s["n_escaped"] + s["n_stuck"] == n + 2 * s["n_pair"]
    assert s["n_photons"] == n and s["e_source"] == pytest.approx(6.0 * n, rel=1e-6)


def test_primary_histories_unchanged_and_secondaries_only_add():
    g = lead_slab(10.0)
    n = 3000
    r0 = oracle.OracleGeometry(g).transport(src(6.0), 3, n, 64, per_photon=True)
    r1 = oracle.OracleGeometry(g, secondaries=1).transport(src(6.0), 3, n, 64, per_photon=True)
    changed = r0["hash"] != r1["hash"]
    assert changed.sum() == r0["stats"]["n_pair"] == r1["stats"]["n_pair"]      # exactly the histories that end in a pair event
    assert np.array_equal(r0["nsteps"][~changed], r1["nsteps"][~changed])
    assert np.array_equal(r0["efinal"], r1["efinal"])                           # the primary's own energy at its end
    assert np.all(r0["efinal"][changed] > 2 * ME_C2)
    assert np.all(r1["nsteps"][changed] >= r0["nsteps"][changed])
    # the annihilation photons carry 2 me c^2 per pair away from the vertex: less is deposited, more escapes
    assert r1["edep"].sum() < r0["edep"].sum()
    assert r1["stats"]["e_escaped"] > r0["stats"]["e_escaped"]
    # below the pair threshold the option changes nothing
    a = oracle.OracleGeometry(g).transport(src(1.0), 3, 500, 64, per_photon=True)
    b = oracle.OracleGeometry(g, secondaries=1).transport(src(1.0), 3, 500, 64, per_photon=True)
    assert np.array_equal(a["hash"], b["hash"]) and np.array_equal(a["edep"], b["edep"])


def test_annihilation_line_from_a_thin_foil():
    """A 0.02 mm lead foil: nearly every annihilation photon leaves without interacting, so the energy the extra
    escaping photons carry is me c^2 each (within the few that scatter first), and never more."""
    g = lead_slab(0.01)
    n = 400000
    r0 = oracle.OracleGeometry(g).transport(src(20.0), 9, n, 64)["stats"]
    r1 = oracle.OracleGeometry(g, secondaries=1).transport(src(20.0), 9, n, 64)["stats"]
    extra_n = r1["n_escaped"] - r0["n_escaped"]
    extra_e = r1["e_escaped"] - r0["e_escaped"]
    assert r1["n_pair"] > 200 and extra_n > 1.9 * r1["n_pair"]
    assert 0.97 * ME_C2 < extra_e / extra_n <= ME_C2 * (1 + 1e-12)


def test_back_to_back_seen_in_four_walls():
    """A thin lead rod on the beam axis inside a square tunnel of four thick lead walls (open along the beam).
    The two annihilation photons of one pair event fly in opposite directions from (nearly) the axis, so when two
    walls light up in one history they are opposite walls; independent directions would give opposite walls in only
    1/3 of the two-wall cases."""
    b = _Builder("four_walls")
    world = b.place(-1, b.box(1000.0, 1000.0, 1000.0), "vacuum")
    b.place(world, b.box(0.25, 0.25, 4.0), "lead")                               # node 1: target rod
    wall_x, wall_y = b.box(50.0, 150.0, 900.0), b.box(50.0, 50.0, 900.0)
    walls = [b.place(world, wall_x, "lead", T=(150.0, 0, 0)), b.place(world, wall_x, "lead", T=(-150.0, 0, 0)),
             b.place(world, wall_y, "lead", T=(0, 150.0, 0)), b.place(world, wall_y, "lead", T=(0, -150.0, 0))]
    g = b.finish()
    og1 = oracle.OracleGeometry(g, secondaries=1)
    n = 6000
    whole = og1.transport(src(8.0), 21, n, 64, per_photon=True)
    h0 = oracle.OracleGeometry(g).transport(src(8.0), 21, n, 64, per_photon=True)["hash"]
    pair_ids = np.nonzero(whole["hash"] != h0)[0]
    assert len(pair_ids) > 300
    opposite = adjacent = 0
    for i in pair_ids:
        e = og1.transport(src(8.0), 21, 1, 64, first_id=int(i))["edep"][walls]
        lit = e > 0
        if lit.sum() == 2:
            if (lit[0] and lit[1]) or (lit[2] and lit[3]):
                opposite += 1
            else:
                adjacent += 1
    assert opposite > 100
    assert adjacent < 0.15 * opposite            # adjacent pairs only through scattering between walls
