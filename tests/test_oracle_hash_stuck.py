"""Pins for the two parts of the oracle that SURVEY 8(c)'s pin table left "parity unpinned": the history hash
(C9: FNV-1a-64 over the little-endian words (vol_before, event) of every step) and the stuck guard (C9: a step of
length <= delta increments a counter, a longer one resets it; at stuck_limit the photon is killed AFTER the step's
event -- DESIGN.md reading 7 -- with n_stuck / E_stuck book-keeping and event word 6).

Hash: the published FNV-1a-64 test vectors (Fowler / Noll / Vo reference vectors: "" , "a", "foobar") through the
oracle's own byte step, and histories known by construction, their expected hash recomputed here from the definition.
Stuck guard: a homogeneous world so large against its surface tolerance that every step is an interaction step of
length s_int <= delta; the expected step counts, fates, energies and hashes follow from the rule alone, and the first
step length is recomputed from the photon's own first uniform (oracle.draw pinned against cuRAND's generator elsewhere).
Also here: the operation counter and the deposit-count tally must not change what the oracle computes."""
import math

import numpy as np
import pytest

import oracle
from paper_1209_5235_b200 import workloads as W
from paper_1209_5235_b200.workloads import _Builder

EV_BOUNDARY, EV_PE, EV_COMPTON, EV_PAIR, EV_CUT, EV_ESCAPE, EV_STUCK = range(7)
FNV_OFFSET, FNV_PRIME, M64 = 0xCBF29CE484222325, 0x100000001B3, (1 << 64) - 1


def fnv1a(data: bytes) -> int:
    """FNV-1a, 64 bit, written from its definition (test-side)."""
    h = FNV_OFFSET
    for b in data:
        h = ((h ^ b) * FNV_PRIME) & M64
    return h


def expected_hash(steps) -> int:
    """steps = [(vol_before, event), ...] -> hash of the little-endian 32-bit words."""
    data = b"".join(int(v & 0xFFFFFFFF).to_bytes(4, "little") + int(e).to_bytes(4, "little") for v, e in steps)
    return fnv1a(data)


# ---- hash ---------------------------------------------------------------------------------------------------------
def test_fnv1a_published_vectors():
    # reference vectors of the FNV-1a 64-bit hash (isthe.com/chongo/tech/comp/fnv test suite): "", "a", "b", "foobar"
    assert oracle.fnv1a_bytes(b"") == 0xCBF29CE484222325
    assert oracle.fnv1a_bytes(b"a") == 0xAF63DC4C8601EC8C
    assert oracle.fnv1a_bytes(b"b") == 0xAF63DF4C8601F1A5
    assert oracle.fnv1a_bytes(b"foobar") == 0x85944171F73967E8
    assert fnv1a(b"foobar") == 0x85944171F73967E8                 # the test-side restatement meets the same vectors


def test_history_words_are_hashed_little_endian_in_order():
    rng = np.random.default_rng(4)
    assert oracle.history_hash([]) == FNV_OFFSET
    assert oracle.history_hash([0x61]) == oracle.fnv1a_bytes(b"a\0\0\0")
    assert oracle.history_hash([0x04030201]) == oracle.fnv1a_bytes(bytes([1, 2, 3, 4]))
    for _ in range(20):
        w = rng.integers(0, 1 << 32, size=rng.integers(1, 40), dtype=np.uint64)
        data = b"".join(int(x).to_bytes(4, "little") for x in w)
        assert oracle.history_hash(w) == fnv1a(data) == oracle.fnv1a_bytes(data)
    assert oracle.history_hash([1, 2]) != oracle.history_hash([2, 1])                 # order matters
    assert oracle.history_hash([0xFFFFFFFF, 5]) == expected_hash([(-1, 5)])           # volume -1 is the word 0xffffffff


def vacuum_world(inner=False):
    b = _Builder("vacuum_world")
    w = b.place(-1, b.box(100.0, 100.0, 100.0), "vacuum")
    if inner:
        b.place(w, b.box(10.0, 10.0, 10.0), "vacuum")
    return b.finish()


def pencil(E, origin=(0.0, 0.0, -50.0)):
    return W.Source(W.SRC_PENCIL, origin, (0.0, 0.0, 1.0), W.E_MONO, E)


@pytest.mark.parametrize("precision", [64, 32])
def test_hash_of_histories_known_by_construction(precision):
    # (1) empty world: one step, (world, ESCAPE)
    r = oracle.OracleGeometry(vacuum_world()).transport(pencil(1.0), 1, 5, precision, per_photon=True)
    assert np.all(r["hash"] == np.uint64(expected_hash([(0, EV_ESCAPE)]))) and np.all(r["nsteps"] == 1)
    assert r["stats"]["n_escaped"] == 5 and r["stats"]["n_steps"] == 5
    # (2) a vacuum box inside: world -> box -> world -> out
    r = oracle.OracleGeometry(vacuum_world(True)).transport(pencil(1.0), 1, 5, precision, per_photon=True)
    assert np.all(r["hash"] == np.uint64(expected_hash([(0, EV_BOUNDARY), (1, EV_BOUNDARY), (0, EV_ESCAPE)]))) and np.all(r["nsteps"] == 3)
    # (3) photon born outside the world: no step at all, the hash is the offset basis
    r = oracle.OracleGeometry(vacuum_world()).transport(pencil(1.0, (0.0, 0.0, -500.0)), 1, 3, precision, per_photon=True)
    assert np.all(r["hash"] == np.uint64(FNV_OFFSET)) and np.all(r["nsteps"] == 0) and r["stats"]["n_escaped"] == 3
    # (4) config 1's geometry under 50 keV photons: world (air) -> lead box -> photoelectric absorption for every photon
    # whose energy never changed (no Compton before): exactly two steps, (world, BOUNDARY), (lead, PE)
    geom = W.slab_geometry(1)
    r = oracle.OracleGeometry(geom).transport(pencil(0.05, (0.0, 0.0, -500.0)), 1, 2000, precision, per_photon=True)
    direct = (r["nsteps"] == 2) & (r["efinal"] == np.float32(0.05) if precision == 32 else r["efinal"] == 0.05)
    assert direct.mean() > 0.9
    assert np.all(r["hash"][direct] == np.uint64(expected_hash([(0, EV_BOUNDARY), (1, EV_PE)])))
    assert np.all(r["hash"][~direct] != np.uint64(expected_hash([(0, EV_BOUNDARY), (1, EV_PE)])))


def test_golden_hashes_follow_from_the_definition():
    """Every photon of config 1 whose history is boundary steps only (it escaped without interacting) went world -> lead
    [-> water -> lead]* -> world -> out; with one water box at most on the beam axis the two possible word lists are known."""
    wl = W.config(1)
    r = oracle.OracleGeometry(wl.geometry).transport(wl.source, wl.seed, 4000, 64, per_photon=True)
    untouched = (r["efinal"] == 1.0) & (r["nsteps"] == 3)
    assert untouched.sum() > 5
    assert np.all(r["hash"][untouched] == np.uint64(expected_hash([(0, EV_BOUNDARY), (1, EV_BOUNDARY), (0, EV_ESCAPE)])))


# ---- stuck guard ----------------------------------------------------------------------------------------------------
def big_water():
    b = _Builder("big_water")
    b.place(-1, b.box(1e7, 1e7, 1e7), "water")
    return b.finish()


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("limit", [1, 3])
def test_every_step_short_by_construction(precision, limit):
    """tol = 1e6 mm in a 2e7 mm water world: every step is an interaction step of ~1e2 mm <= delta = 5e5 mm.  A photon
    is stuck after exactly `limit` steps unless it was absorbed first; the stuck test comes after the step's event, so the
    Compton scatter of the last step has happened (deposit tallied, energy lowered) and its event word is STUCK."""
    n = 2000
    opts = dict(stuck_limit=limit, **({"tol64": 1e6} if precision == 64 else {"tol32": 1e6}))
    r = oracle.OracleGeometry(big_water(), **opts).transport(pencil(1.0, (0.0, 0.0, 0.0)), 7, n, precision, per_photon=True)
    s = r["stats"]
    absorbed = s["n_pe"] + s["n_pair"] + s["n_cut"]
    assert s["n_escaped"] == 0 and s["n_stuck"] == n - absorbed and absorbed <= 20
    stuck_hash = np.uint64(expected_hash([(0, EV_COMPTON)] * (limit - 1) + [(0, EV_STUCK)]))
    is_stuck = r["hash"] == stuck_hash
    assert is_stuck.sum() == s["n_stuck"]
    assert np.all(r["nsteps"][is_stuck] == limit) and np.all(r["nsteps"][~is_stuck] <= limit)
    assert s["n_steps"] == int(r["nsteps"].sum())
    assert s["n_compton"] == s["n_steps"] - s["n_pe"] - s["n_pair"]                   # the last step's scatter did happen
    assert np.all(r["efinal"][is_stuck] < 1.0)
    rel = 1e-12 if precision == 64 else 1e-5
    assert abs(s["e_stuck"] - r["efinal"][is_stuck].sum()) <= rel * s["e_source"]
    assert abs(s["e_stuck"] - (s["e_source"] - r["edep"].sum())) <= rel * s["e_source"]    # E_stuck = E_source - edep
    assert abs(r["edep"].sum() - s["e_deposited"]) <= rel * s["e_source"]


def test_counter_resets_after_a_long_step_and_uses_the_step_length():
    """delta = one mean free path: a photon is killed at its second consecutive step of length <= delta.  The first step
    length is recomputed here: s_1 = -ln(U_0) / mu(water, 1 MeV) with U_0 the photon's own first uniform."""
    n, seed, limit = 4000, 11, 2
    og0 = oracle.OracleGeometry(big_water())
    mu = float(og0.mu(0, 1.0, 64).sum())
    delta = 1.0 / mu
    og = oracle.OracleGeometry(big_water(), tol64=2.0 * delta, stuck_limit=limit)
    assert og.tolerance(64) == 2.0 * delta
    r = og.transport(pencil(1.0, (0.0, 0.0, 0.0)), seed, n, 64, per_photon=True)
    s1 = np.array([-math.log(oracle.draw(seed, i, 0, 64)) / mu for i in range(n)])
    short1 = s1 <= delta
    stuck_at_2 = (r["nsteps"] == 2) & (r["hash"] == np.uint64(expected_hash([(0, EV_COMPTON), (0, EV_STUCK)])))
    assert not np.any(stuck_at_2 & ~short1)                       # a long first step resets: nobody is stuck at step 2 after it
    assert abs(short1.mean() - (1 - math.exp(-1))) < 0.03
    frac = stuck_at_2[short1].mean()                              # P(s_2 <= delta) at the lower energy after one scatter: >= 1 - 1/e
    assert 0.60 < frac < 0.90
    later = (r["nsteps"] > 2)
    assert later.sum() > 500 and r["stats"]["n_stuck"] > 0.9 * n
    # nobody can be stuck after one step when limit = 2
    assert not np.any(r["nsteps"] < 2) or r["stats"]["n_pe"] > 0


def test_default_limit_is_not_reached_in_the_standard_configs():
    wl = W.config(1)
    r = oracle.OracleGeometry(wl.geometry).transport(wl.source, wl.seed, 3000, 64)
    assert r["stats"]["n_stuck"] == 0 and r["stats"]["e_stuck"] == 0.0


def test_zero_length_boundary_steps_in_a_coarse_tolerance_phantom():
    """Boundary steps of length <= delta arise by themselves when the tolerance is a sizeable fraction of the voxel
    size (direction changes next to a face, entries snapped to 0): with stuck_limit 1 and 2 some photons are killed, the
    book-keeping still closes and the killed photons' last event word is STUCK."""
    g = W.phantom_geometry(16, 2.0, 3); src = W.phantom_source(16, half_angle_deg=0.8)
    for limit in (1, 2):
        r = oracle.OracleGeometry(g, tol64=0.4, stuck_limit=limit).transport(src, 3, 5000, 64, per_photon=True)
        s = r["stats"]
        assert s["n_stuck"] > 5 and s["e_stuck"] > 0
        assert s["n_pe"] + s["n_pair"] + s["n_cut"] + s["n_escaped"] + s["n_stuck"] == 5000
        assert abs((r["edep"].sum() + s["e_escaped"] + s["e_stuck"]) / s["e_source"] - 1) < 1e-12
    r8 = oracle.OracleGeometry(g, tol64=0.4, stuck_limit=8).transport(src, 3, 5000, 64)
    assert r8["stats"]["n_stuck"] == 0


# ---- operation counter and deposit tally leave the computation alone ------------------------------------------------
@pytest.mark.parametrize("k", [1, 2, 3, 4])
def test_operation_counter_follows_the_fp64_histories(k):
    wl = W.config(k)
    og = oracle.OracleGeometry(wl.geometry)
    n = 1500
    counts, st = og.transport_count_ops(wl.source, wl.seed, n)
    ref = og.transport(wl.source, wl.seed, n, 64)["stats"]
    for key in ("n_steps", "n_compton", "n_pe", "n_pair", "n_cut", "n_escaped", "n_stuck"):
        assert st[key] == ref[key], key
    assert abs(st["e_deposited"] - ref["e_deposited"]) <= 1e-12 * ref["e_source"]
    per_step = counts["flops"] / st["n_steps"]
    assert counts["flops"] == sum(counts[c] for c in ("add", "mul", "div", "sqrt", "cmp", "trans")) + 2 * counts["fma"]
    # a ComputeStep is at least one transform of point and direction (6 fma + ...) and one DistanceToOut
    assert 100 < per_step < 5000, per_step
    # counts are additive over photon-id ranges (up to the one division tol / 2 of a run's set-up)
    c1, s1 = og.transport_count_ops(wl.source, wl.seed, 700)
    c2, s2 = og.transport_count_ops(wl.source, wl.seed, n - 700, first_id=700)
    assert c1["flops"] + c2["flops"] == counts["flops"] + 1 and s1["n_steps"] + s2["n_steps"] == st["n_steps"]


def test_operation_counter_on_navigation_queries():
    wl = W.config(5)
    og = oracle.OracleGeometry(wl.geometry)
    pos, d = W.nav_queries(wl.geometry, 4000, seed=wl.seed)
    c = og.nav_count_ops(pos, d)
    assert 200 < c["flops"] / 4000 < 5000
    # one box world, a point well inside, an axis-parallel ray: locate = 1 transform + 1 Inside, step = 2 transforms + 1 DistanceToOut
    g = vacuum_world()
    c = oracle.OracleGeometry(g).nav_count_ops(np.array([[1.0, 2.0, 3.0]]), np.array([[0.0, 0.0, 1.0]]))
    # locate: point transform (3 sub, 3 mul, 6 fma) + Inside (3 abs, 3 sub, 2 max, <= 2 compares); step: point + direction
    # transforms (3 sub, 6 mul, 12 fma), DistanceToOut (compares and one division on the moving axis), best > max_step,
    # the move (3 fma), relocate at the exit point = point transform + Inside (surface) + direction transform + DistanceToOut (0, no division)
    assert c["fma"] == 6 + 12 + 3 + 12 and c["div"] == 1 and c["sqrt"] == 0 and c["trans"] == 0


def test_deposit_tally_counts_and_squares():
    wl = W.config(1)
    og = oracle.OracleGeometry(wl.geometry)
    a = og.transport(wl.source, wl.seed, 3000, 64, tally=True)
    b = og.transport(wl.source, wl.seed, 3000, 64)
    assert np.array_equal(a["edep"], b["edep"])
    s = a["stats"]
    assert int(a["n_dep"].sum()) == s["n_pe"] + s["n_compton"] + s["n_pair"]
    assert np.all((a["n_dep"] == 0) == (a["edep_sq"] == 0))
    nz = a["n_dep"] > 0
    # Cauchy-Schwarz per volume: (sum d)^2 <= n sum d^2, and every deposit is at most the source energy
    assert np.all(a["edep"][nz] ** 2 <= a["n_dep"][nz] * a["edep_sq"][nz] * (1 + 1e-12))
    assert np.all(a["edep_sq"][nz] <= a["edep"][nz] * 1.0 * (1 + 1e-12))
