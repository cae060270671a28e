"""Pins for the rest of SURVEY 8(f) NEXT-3 in the oracle: Rayleigh (coherent) scattering and the tabulated photoelectric
coefficient (readings 18 and 19; both are options, the default physics is BASELINE.json config 1's).

Rayleigh: the angular density 1 + cos^2(theta) has closed-form moments and CDF; the scatter keeps the energy and deposits
nothing; mu_R scales as n Z^2 / E^2 by definition; its normalisation is a calibration (the model's mu/rho of aluminium at
1 MeV then equals the value the paper prints) and therefore stays "parity unpinned".
Table: generated from the closed form, it must reproduce the Z^5 / E^3.5 law to the interpolation error of the grid, be
exact at grid nodes, clamp at the ends, and show the K jump of lead where the edge model puts it."""
import math

import numpy as np
import pytest
from scipy import stats

import oracle
from paper_1209_5235_b200 import workloads as W
from paper_1209_5235_b200.workloads import _Builder

EV_BOUNDARY, EV_PE, EV_COMPTON, EV_PAIR, EV_CUT, EV_ESCAPE, EV_STUCK, EV_RAYLEIGH = range(8)


def expected_hash(steps) -> int:
    """FNV-1a-64 over the little-endian 32-bit words (vol_before, event) of every step, from the definition (S:C9)."""
    h = 0xCBF29CE484222325
    for v, e in steps:
        for b in int(v & 0xFFFFFFFF).to_bytes(4, "little") + int(e).to_bytes(4, "little"):
            h = ((h ^ b) * 0x100000001B3) & ((1 << 64) - 1)
    return h


def one_material_world(material, half=100.0):
    b = _Builder("one_" + material)
    b.place(-1, b.box(half, half, half), material)
    return b.finish()


def pencil(E, z0=0.0):
    return W.Source(W.SRC_PENCIL, (0.0, 0.0, z0), (0.0, 0.0, 1.0), W.E_MONO, E)


# ---- Rayleigh ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", [64, 32])
def test_rayleigh_angle_follows_one_plus_cos_squared(precision):
    c, nt = oracle.rayleigh_sample(5, 200000, precision)
    assert np.all(np.abs(c) <= 1.0)
    # moments of p(c) = (3/8)(1 + c^2): <c> = 0, <c^2> = 2/5, <c^4> = (2/5 + 2/7) / (8/3) = 9/35
    assert abs(c.mean()) < 4e-3 and abs((c ** 2).mean() - 0.4) < 3e-3 and abs((c ** 4).mean() - 9.0 / 35.0) < 3e-3
    cdf = lambda t: 0.375 * (t + t ** 3 / 3.0) + 0.5
    assert stats.kstest(c[:50000], cdf).pvalue > 1e-3
    assert abs(nt.mean() - 1.5) < 0.01                           # acceptance 2/3: the envelope is 2, the mean of 1 + c^2 is 4/3


def test_rayleigh_coefficient_definition_and_calibration():
    og_al = oracle.OracleGeometry(one_material_world("aluminium"), rayleigh=1)
    og_pb = oracle.OracleGeometry(one_material_world("lead"), rayleigh=1)
    assert oracle.OracleGeometry(one_material_world("aluminium")).mu_rayleigh(0, 1.0) == 0.0          # off by default
    m1, m2 = og_al.mu_rayleigh(0, 1.0), og_al.mu_rayleigh(0, 0.1)
    assert abs(m2 / m1 - 100.0) < 1e-9                           # 1 / E^2
    Z, A, rho = W.MATERIALS["aluminium"]; Zp, Ap, rhop = W.MATERIALS["lead"]
    assert abs(og_pb.mu_rayleigh(0, 1.0) / m1 - (rhop / Ap * Zp ** 2) / (rho / A * Z ** 2)) < 1e-9 * 1e3      # n Z^2
    # normalisation: 7.886e-3 barn per aluminium atom at 1 MeV, chosen so that the model's total mu / rho of aluminium at
    # 1 MeV is the paper's 0.06146 cm^2/g -- a calibration, not an independent check
    assert abs(m1 - rho * 6.02214076e23 / A * 7.886e-3 * 1e-24 / 10.0) < 1e-12 * m1 * 1e3
    total = (og_al.mu(0, 1.0).sum() + m1) * 10.0 / rho
    assert abs(total - 0.06146) < 2e-6
    og_big = oracle.OracleGeometry(one_material_world("aluminium"), rayleigh=1, sigma_r0=1.0)
    assert abs(og_big.mu_rayleigh(0, 1.0) / m1 - 1.0 / 7.886e-3) < 1e-9 * 200


@pytest.mark.parametrize("precision", [64, 32])
def test_rayleigh_scatter_keeps_the_energy_and_deposits_nothing(precision):
    """A cross-section so large that nearly every interaction is a Rayleigh scatter (5e4 x Compton, in air so that the free path stays millimetres): photons that only scattered
    coherently leave with their source energy and deposit nothing, and a photon with exactly one scatter has the history
    (world, RAYLEIGH), (world, ESCAPE)."""
    n = 4000
    og = oracle.OracleGeometry(one_material_world("air", 5.0), rayleigh=1, sigma_r0=2.5e5)      # mean free path 2.6 mm in a 10 mm world of thin air
    r = og.transport(pencil(1.0), 9, n, precision, per_photon=True)
    s = r["stats"]
    assert s["n_rayleigh"] > 2 * n and s["n_pe"] + s["n_pair"] + s["n_cut"] <= 5
    assert s["n_rayleigh"] + s["n_compton"] + s["n_pe"] + s["n_pair"] + s["n_escaped"] == s["n_steps"]
    pure = r["efinal"] == (1.0 if precision == 64 else np.float32(1.0))
    assert pure.mean() > 0.99
    assert r["edep"].sum() <= (n - pure.sum()) * 1.0 + 1e-9      # only the few Compton / PE events deposit
    one = pure & (r["nsteps"] == 2)
    assert one.any() and np.all(r["hash"][one] == np.uint64(expected_hash([(0, EV_RAYLEIGH), (0, EV_ESCAPE)])))
    two = pure & (r["nsteps"] == 3)
    assert two.any() and np.all(r["hash"][two] == np.uint64(expected_hash([(0, EV_RAYLEIGH), (0, EV_RAYLEIGH), (0, EV_ESCAPE)])))
    assert abs((r["edep"].sum() + s["e_escaped"] + s["e_stuck"]) / s["e_source"] - 1) < (1e-12 if precision == 64 else 1e-6)


def test_transmission_with_rayleigh_is_exp_minus_total_mu_x():
    """Unscattered transmission through a slab (Eq. 2-5) with the fourth process switched on."""
    geom = W.homogeneous_slab("lead", half=(500.0, 500.0, 2.5), world_half=1000.0)
    og = oracle.OracleGeometry(geom, rayleigh=1)
    E, n = 0.3, 40000
    mu = og.mu(1, E).sum() + og.mu_rayleigh(1, E)
    assert og.mu_rayleigh(1, E) > 0.03 * mu                      # coherent scattering matters here
    r = og.transport(pencil(E, -100.0), 4, n, 64, per_photon=True)
    untouched = (r["nsteps"] == 3) & (r["efinal"] == E)          # world -> slab -> world -> out without an event ... or Rayleigh only
    straight = r["hash"] == np.uint64(expected_hash([(0, EV_BOUNDARY), (1, EV_BOUNDARY), (0, EV_ESCAPE)]))
    p = math.exp(-mu * 5.0)
    assert abs(straight.mean() - p) < 4 * math.sqrt(p * (1 - p) / n)
    assert r["stats"]["n_rayleigh"] > 0 and untouched.sum() >= straight.sum()


def test_default_physics_is_unchanged_and_the_option_is_additive():
    wl = W.config(1)
    a = oracle.OracleGeometry(wl.geometry).transport(wl.source, wl.seed, 2000, 64, per_photon=True)
    b = oracle.OracleGeometry(wl.geometry, rayleigh=0, pe_table_per_decade=0).transport(wl.source, wl.seed, 2000, 64, per_photon=True)
    assert np.array_equal(a["hash"], b["hash"]) and a["stats"]["n_rayleigh"] == 0
    c = oracle.OracleGeometry(wl.geometry, rayleigh=1).transport(wl.source, wl.seed, 2000, 64, per_photon=True)
    assert c["stats"]["n_rayleigh"] > 0 and (c["hash"] != a["hash"]).mean() > 0.02
    s = c["stats"]
    assert s["n_pe"] + s["n_pair"] + s["n_cut"] + s["n_escaped"] + s["n_stuck"] == 2000
    assert abs((c["edep"].sum() + s["e_escaped"] + s["e_stuck"]) / s["e_source"] - 1) < 1e-12


# ---- tabulated photoelectric coefficient ----------------------------------------------------------------------------------
def test_table_reproduces_the_power_law_it_was_generated_from():
    geom = one_material_world("lead")
    law = oracle.OracleGeometry(geom)
    for P, tol in ((256, 2e-4), (64, 2.5e-3)):
        tab = oracle.OracleGeometry(geom, pe_table_per_decade=P)
        E = np.exp(np.random.default_rng(1).uniform(math.log(0.0101), math.log(990.0), 400))
        rel = np.array([abs(tab.mu(0, e)[0] / law.mu(0, e)[0] - 1) for e in E])
        assert rel.max() < tol, (P, rel.max())
        # interpolation error of a power law E^-3.5 between nodes a step d = ln 10 / P apart: <= (3.5 d)^2 / 8
        assert rel.max() > 0.2 * (3.5 * math.log(10) / P) ** 2 / 8
        for k in (0, 1, P, 3 * P + 7, 5 * P):                     # exact at the nodes (up to the rounding of ln / pow)
            e = 0.01 * 10 ** (k / P)
            assert abs(tab.mu(0, e)[0] / law.mu(0, e)[0] - 1) < (1e-6 if k < 5 * P else 1e-5)      # the top node is approached from just below (clamp)
        assert tab.mu(0, 5000.0)[0] == tab.mu(0, 999.9999999)[0] or abs(tab.mu(0, 5000.0)[0] / tab.mu(0, 1000.0)[0] - 1) < 1e-3      # clamped
        assert abs(tab.mu(0, 0.001)[0] / tab.mu(0, 0.01)[0] - 1) < 1e-6
        assert np.array_equal(tab.mu(0, 1.0)[1:], law.mu(0, 1.0)[1:])                                # Compton and pair untouched
    with pytest.raises(RuntimeError):
        oracle.OracleGeometry(geom, pe_table_per_decade=5000)


def test_k_edge_model_of_lead():
    geom = one_material_world("lead")
    flat = oracle.OracleGeometry(geom, pe_table_per_decade=256)
    edge = oracle.OracleGeometry(geom, pe_table_per_decade=256, pe_k_edge=1)
    eK = 13.6e-6 * 81.0 ** 2                                     # 89.2 keV
    assert 0.085 < eK < 0.092
    above, below = eK * 1.03, eK * 0.97
    assert abs(edge.mu(0, above)[0] / flat.mu(0, above)[0] - 1) < 1e-9
    assert abs(edge.mu(0, below)[0] / flat.mu(0, below)[0] - 0.2) < 1e-9           # jump ratio 5
    assert edge.mu(0, below)[0] < edge.mu(0, above)[0]                             # absorption rises across the edge
    E = np.geomspace(0.011, 900.0, 300)
    m = np.array([edge.mu(0, e)[0] for e in E])
    falling = np.diff(m) < 0
    assert (~falling).sum() <= 2                                                    # monotone except the one interval with the edge
    # materials whose K edge lies below the 10 keV cut are untouched
    gw = one_material_world("water")
    assert np.array_equal(oracle.OracleGeometry(gw, pe_table_per_decade=64, pe_k_edge=1).mu(0, 0.05), oracle.OracleGeometry(gw, pe_table_per_decade=64).mu(0, 0.05))


def test_transport_with_the_table_stays_close_to_the_closed_form():
    wl = W.config(1)
    a = oracle.OracleGeometry(wl.geometry).transport(wl.source, wl.seed, 4000, 64, per_photon=True)
    b = oracle.OracleGeometry(wl.geometry, pe_table_per_decade=256).transport(wl.source, wl.seed, 4000, 64, per_photon=True)
    same = (a["hash"] == b["hash"]) & (a["nsteps"] == b["nsteps"])
    assert same.mean() > 0.99                                     # mu_PE moves by < 2e-4 relative: a handful of process choices flip
    s = b["stats"]
    assert abs((b["edep"].sum() + s["e_escaped"] + s["e_stuck"]) / s["e_source"] - 1) < 1e-12
    # with the edge, 60 keV photons in lead are absorbed five times less often by the photoelectric effect
    geom = W.homogeneous_slab("lead", half=(500.0, 500.0, 0.0005), world_half=1000.0)      # 1 um of lead: absorption still linear in mu
    src = W.Source(W.SRC_PENCIL, (0.0, 0.0, -100.0), (0.0, 0.0, 1.0), W.E_MONO, 0.06)
    flat = oracle.OracleGeometry(geom, pe_table_per_decade=256).transport(src, 3, 20000, 64)["stats"]
    edge = oracle.OracleGeometry(geom, pe_table_per_decade=256, pe_k_edge=1).transport(src, 3, 20000, 64)["stats"]
    assert 3.5 * edge["n_pe"] < flat["n_pe"] < 7.0 * edge["n_pe"] and edge["n_pe"] > 50
