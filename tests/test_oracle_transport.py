"""Pins for the oracle's transport loop (Algorithm 1 L55-76, Eq. 2-7).
BASELINE.json north_star: "unscattered slab transmission exp(-mu x)"."""
import json
import math
import os

import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_1209_5235_b200 import workloads as W

ME, RE, NA, ALPHA = 0.51099895, 2.8179403262e-13, 6.02214076e23, 7.2973525693e-3
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def mu_independent(name, E):
    """total linear attenuation [1/mm] written out from the definitions (quadrature for Compton)."""
    Z, A, rho = W.MATERIALS[name]
    k = E / ME

    def dsde(eps):
        t = (1 - eps) / (k * eps)
        return math.pi * RE * RE / k * (1 / eps + eps) * (1 - eps * t * (2 - t) / (1 + eps * eps))
    kn, _ = integrate.quad(dsde, 1 / (1 + 2 * k), 1.0, epsrel=1e-12)
    pe = 1750e-24 * (Z / 82) ** 5 * (0.1 / E) ** 3.5
    pair = 0.0
    if k > 2:
        pair = ALPHA * RE * RE * Z * Z * max(0.0, min(28 / 9 * math.log(2 * k) - 218 / 27, 28 / 9 * math.log(183 * Z ** (-1 / 3)) - 2 / 27))
    return rho * NA / A * (pe + Z * kn + pair) / 10


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("material,E,half_z", [("water", 1.0, 50.0), ("lead", 10.0, 5.0), ("bone", 0.2, 20.0)])
def test_unscattered_slab_transmission(material, E, half_z, precision):
    """Eq. 2/3/5: the fraction of photons crossing a homogeneous slab of thickness x with no interaction is
    exp(-mu x).  Unscattered photons are exactly those with 3 steps (enter, leave, escape) and E unchanged."""
    geom = W.homogeneous_slab(material, half=(1000.0, 1000.0, half_z))
    og = oracle.OracleGeometry(geom)
    src = W.Source(W.SRC_PENCIL, (0, 0, -500.0), (0, 0, 1.0), W.E_MONO, E)
    n = 200000
    r = og.transport(src, seed=11, n=n, precision=precision, per_photon=True)
    unsc = np.sum((r["nsteps"] == 3) & (r["efinal"] == (float(np.float32(E)) if precision == 32 else E)))
    p = math.exp(-mu_independent(material, E) * 2 * half_z)
    sigma = math.sqrt(n * p * (1 - p))
    assert abs(unsc - n * p) < 4 * sigma, (unsc, n * p, sigma)
    s = r["stats"]
    assert s["n_stuck"] == 0 and s["n_photons"] == n


def test_free_path_distribution_across_layers():
    """Eq. 5-7 with piecewise-constant mu: in the calorimeter stack the depth of the FIRST interaction
    follows P(T < t) = 1 - exp(-G(t)); check the per-layer first-interaction counts (KS-style, chi^2)."""
    geom = W.calorimeter_geometry(n_pairs=6)
    og = oracle.OracleGeometry(geom)
    src = W.Source(W.SRC_PENCIL, (0, 0, -500.0), (0, 0, 1.0), W.E_MONO, 10.0)
    n = 100000
    # photons that die in their first interaction (PE or pair) deposit their full energy in that layer:
    # pick those by efinal == 10 and nsteps == (layers crossed + 3); layer of death = from nsteps
    r = og.transport(src, seed=5, n=n, precision=64, per_photon=True)
    mu_pb, mu_sc, mu_air = (mu_independent(m, 10.0) for m in ("lead", "scint", "air"))
    # survival to the front of the stack through 500-21 mm of air in world + mother
    hz = 6 * 7 / 2
    G = mu_air * (500 - hz)
    # a photon whose first interaction happens in layer j (0-based) has taken exactly j + 2 steps at that point
    # (world -> layer 0 directly, because the mother's front face coincides with layer 0's: relocate descends;
    # j layer crossings; the interaction step).  Count photons absorbed at the first interaction
    # (efinal == 10, not escaped): nsteps = j + 2
    dead_first = (r["efinal"] == 10.0) & (r["nsteps"] >= 2) & (r["nsteps"] <= 13)
    exp_first = []
    for j in range(12):
        mu = mu_pb if j % 2 == 0 else mu_sc
        t = 2.0 if j % 2 == 0 else 5.0
        p_int = math.exp(-G) * (1 - math.exp(-mu * t))
        G += mu * t
        exp_first.append(p_int)
    # fraction of first interactions that are absorbing (PE + pair) in each material
    def absorb_frac(name):
        Z, A, rho = W.MATERIALS[name]
        k = 10.0 / ME
        pe = 1750e-24 * (Z / 82) ** 5 * (0.1 / 10.0) ** 3.5
        pair = ALPHA * RE * RE * Z * Z * max(0.0, min(28 / 9 * math.log(2 * k) - 218 / 27, 28 / 9 * math.log(183 * Z ** (-1 / 3)) - 2 / 27))
        tot = mu_independent(name, 10.0) * 10 / (rho * NA / A)
        return (pe + pair) / tot
    chi2 = 0.0
    for j in range(12):
        obs = np.sum(dead_first & (r["nsteps"] == j + 2))
        # escaping photons also keep efinal == 10 but never have nsteps <= 13 here (they cross all 12 layers: 14 steps)
        exp = n * exp_first[j] * absorb_frac("lead" if j % 2 == 0 else "scint")
        chi2 += (obs - exp) ** 2 / exp
    assert chi2 < 40.0, chi2        # 12 dof, p ~ 1e-4


@pytest.mark.parametrize("precision", [64, 32])
def test_energy_bookkeeping(precision):
    for k, n in ((1, 5000), (2, 2000)):
        wl = W.config(k)
        og = oracle.OracleGeometry(wl.geometry)
        r = og.transport(wl.source, wl.seed, n, precision)
        s = r["stats"]
        total = r["edep"].sum() + s["e_escaped"] + s["e_stuck"]
        assert abs(total / s["e_source"] - 1) < (1e-12 if precision == 64 else 2e-6)
        assert abs(r["edep"].sum() - s["e_deposited"]) <= 1e-9 * s["e_source"]
        assert s["n_pe"] + s["n_pair"] + s["n_cut"] + s["n_escaped"] + s["n_stuck"] == n
        assert s["n_stuck"] == 0


def test_order_independence_and_sharding():
    """PAPER.md L156-158 test idea: results do not depend on launch order -- photon i is a function of
    (seed, i) only, so disjoint id ranges add up to the whole run."""
    wl = W.config(1)
    og = oracle.OracleGeometry(wl.geometry)
    whole = og.transport(wl.source, 1, 3000, 64, per_photon=True)
    a = og.transport(wl.source, 1, 1000, 64, first_id=0, per_photon=True)
    b = og.transport(wl.source, 1, 2000, 64, first_id=1000, per_photon=True)
    assert np.array_equal(whole["hash"], np.concatenate([a["hash"], b["hash"]]))
    assert np.array_equal(whole["nsteps"], np.concatenate([a["nsteps"], b["nsteps"]]))
    assert np.allclose(whole["edep"], a["edep"] + b["edep"], rtol=1e-12, atol=0)
    assert not np.array_equal(whole["hash"], og.transport(wl.source, 2, 3000, 64, per_photon=True)["hash"])


@pytest.mark.parametrize("precision", [64, 32])
def test_grid_navigation_gives_identical_histories(precision):
    n = 8
    geom = W.phantom_geometry(n, 2.0, seed=3, world_half=300.0)
    og = oracle.OracleGeometry(geom)
    src = W.phantom_source(n, 2.0, distance=200.0, half_angle_deg=2.5, energy=0.3)
    a = og.transport(src, 3, 3000, precision, per_photon=True, use_grid=True)
    b = og.transport(src, 3, 3000, precision, per_photon=True, use_grid=False)
    assert np.array_equal(a["hash"], b["hash"]) and np.array_equal(a["edep"], b["edep"])
    assert a["stats"]["n_steps"] > 8 * 3000 and a["stats"]["n_stuck"] == 0
    geom = W.detector_geometry(seed=4, n_phi=8, n_z=8, barrels=((200, 400), (450, 650)))
    og = oracle.OracleGeometry(geom)
    a = og.transport(W.detector_source(), 4, 3000, precision, per_photon=True, use_grid=True)
    b = og.transport(W.detector_source(), 4, 3000, precision, per_photon=True, use_grid=False)
    assert np.array_equal(a["hash"], b["hash"]) and np.array_equal(a["edep"], b["edep"])
    assert a["stats"]["n_stuck"] == 0


def test_fp32_mode_agrees_statistically_with_fp64():
    wl = W.config(2)
    og = oracle.OracleGeometry(wl.geometry)
    n = 20000
    a = og.transport(wl.source, 2, n, 64); b = og.transport(wl.source, 2, n, 32)
    assert abs(a["edep"].sum() / b["edep"].sum() - 1) < 1e-3 + 3 / math.sqrt(n)
    assert abs(a["stats"]["n_steps"] / b["stats"]["n_steps"] - 1) < 0.02
    assert b["stats"]["n_stuck"] == 0


def test_no_stuck_photons_on_touching_voxels_fp32():
    """SURVEY 8(c) C4 evidence re-created: touching voxels hit from 1 m away in fp32, no stuck photons."""
    n = 8
    geom = W.phantom_geometry(n, 2.0, seed=3, world_half=1200.0)
    og = oracle.OracleGeometry(geom)
    src = W.phantom_source(n, 2.0, distance=1056.0, half_angle_deg=0.4, energy=6.0)
    r = og.transport(src, 3, 20000, 32)
    assert r["stats"]["n_stuck"] == 0
    assert r["stats"]["n_steps"] > 8 * 20000


def test_golden_config1():
    """Regression pin written by tests/golden/make_golden.py (oracle only): config 1, fp64, seed 1."""
    with open(os.path.join(GOLDEN, "config1_oracle_fp64.json")) as f:
        gold = json.load(f)
    wl = W.config(1)
    og = oracle.OracleGeometry(wl.geometry)
    r = og.transport(wl.source, wl.seed, gold["n_photons"], 64, per_photon=True)
    for k in ("n_steps", "n_compton", "n_pe", "n_pair", "n_cut", "n_escaped", "n_stuck"):
        assert r["stats"][k] == gold["stats"][k]
    assert np.allclose(r["edep"], gold["edep"], rtol=1e-9)
    assert [int(h) for h in r["hash"][:16]] == gold["hash_first16"]
