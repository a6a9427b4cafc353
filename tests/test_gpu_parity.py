"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Bars (BASELINE.json north_star): spins / flip order / flip counts / neighbour tables
bit-exact; fp64 fields within 1e-12 relative to max|h|."""
import math

import numpy as np
import pytest

from paper_2002_11401_b200 import workloads as W

pytestmark = pytest.mark.gpu

FIELD_TOL = 1e-12


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2002_11401_b200 import binding
    return binding


def mk(B, w, spins=None):
    from oracle import Oracle
    sim = B.Sim(w.pos, w.angle, w.hc, w.params)
    orc = Oracle(w.pos, w.angle, w.hc, w.params, spins=w.spins if spins is None else spins)
    sim.set_spins(w.spins if spins is None else spins)
    if w.sigma_th:
        sim.set_thermal(w.sigma_th, w.thermal_seed); orc.set_thermal(w.sigma_th, w.thermal_seed)
    return sim, orc


def field_err(hg, ho):
    return np.abs(hg - ho).max() / max(np.abs(ho).max(), 1e-300)


def run_parity(B, w, stride=1, tier="B", check_fields_every=0):
    sim, orc = mk(B, w)
    total = 0
    steps = list(enumerate(w.fields))[::stride]
    for n_done, (t, (hx, hy)) in enumerate(steps):
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        n = sim.relax()
        no, log = getattr(orc, "relax_" + tier)()
        assert n == no, (t, n, no)
        if n:
            glog = sim.get_flip_log().cpu().numpy()
            assert np.array_equal(glog, log), f"flip order differs at step {t}"
        total += n
        if check_fields_every and n_done % check_fields_every == 0:
            assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    assert field_err(sim.get_fields(1).cpu().numpy(), orc.fields(1)) < FIELD_TOL
    ev, gap, thr = orc.monitor()
    assert ev == 0, "oracle recorded a near-tie: flip order not well posed on this input"
    assert sim.scan()[0] == 0 and orc.scan()[0] == 0
    return total, sim, orc


# ------------------------------------------------------------------ A1/A2: neighbour tables, couplings
@pytest.mark.parametrize("which,scale", [("1", None), ("2", 12), ("3", 14), ("5", 24)])
def test_neighbor_tables_bit_exact(B, which, scale):
    from oracle import Oracle
    w = W.config(which, scale=scale)
    sim = B.Sim(w.pos, w.angle, w.hc, w.params)
    orc = Oracle(w.pos, w.angle, w.hc, w.params)
    ref = orc.neighbors()
    got = sim.get_neighbors().cpu().numpy()
    assert sim.K == ref.shape[1] and sim.n_interactions == orc.num_interactions
    assert np.array_equal(got, ref)


def test_config2_full_neighbor_count(B):
    w = W.config("2")
    sim = B.Sim(w.pos, w.angle, w.hc, w.params)
    assert (sim.N, sim.K, sim.n_interactions) == (7699, 14, 105476)
    # full size, stencil (the auto choice) against the oracle's direct evaluation on random spins
    from oracle import Oracle
    for which in ("2", "2b"):
        w = W.config(which)
        spins = W.random_spins(w.N, seed=17)
        sim = B.Sim(w.pos, w.angle, w.hc, w.params); sim.set_spins(spins)
        assert sim.lattice()["active"] and sim.lattice()["nsub"] == 3
        orc = Oracle(w.pos, w.angle, w.hc, w.params, spins=spins)
        sim.update_fields()
        assert field_err(sim.get_fields(1).cpu().numpy(), orc.fields(1)) < FIELD_TOL


# ------------------------------------------------------------------ A3: full gather (ELL and lattice stencil)
def _check_all_fields(sim, orc):
    for which_f in (0, 1, 2, 3):
        hg = sim.get_fields(which_f).cpu().numpy(); ho = orc.fields(which_f)
        if np.abs(ho).max() > 0:
            assert np.abs(hg - ho).max() / np.abs(ho).max() < FIELD_TOL, which_f
        else:
            assert np.abs(hg).max() == 0


@pytest.mark.parametrize("variant", ["ell", "stencil"])
@pytest.mark.parametrize("which,scale", [("1", None), ("2", 20), ("3", 30), ("4", 40), ("5", 40)])
def test_full_gather_fields(B, which, scale, variant):
    w = W.config(which, scale=scale)
    spins = W.random_spins(w.N, seed=11)
    sim, orc = mk(B, w, spins=spins)
    lat = sim.lattice()
    if variant == "stencil":
        assert lat["active"], lat                 # every BASELINE geometry is a detected lattice (kagome: 3 sublattices)
        sim.set_gather_variant(B.GATHER_STENCIL)
    else:
        sim.set_gather_variant(B.GATHER_ELL_F64)
    hx, hy = w.fields[len(w.fields) // 3]
    sim.set_field(hx, hy, 3); orc.set_field(hx, hy, 3)
    sim.update_fields()
    _check_all_fields(sim, orc)


def test_lattice_detection_tables(B):
    """Sublattice count (square/pinwheel 2, kagome 3), stencil extents and slot counts."""
    w = W.config("5", scale=24)                       # nd = 10: 316 same + 316 cross sublattice offsets
    sim = B.Sim(w.pos, w.angle, w.hc, w.params)
    lat = sim.lattice()
    assert lat["active"] and (lat["nsub"], lat["Ru"], lat["Rv"]) == (2, 10, 10), lat
    assert lat["slots"] == 4 * 316 and lat["max_dev"] == 0.0
    assert (lat["U"], lat["V"]) == (25, 25)
    w = W.config("1")
    lat = B.Sim(w.pos, w.angle, w.hc, w.params).lattice()
    assert lat["active"] and lat["nsub"] == 2 and lat["slots"] == 16, lat       # 4 same + 4 cross, per sublattice
    w = W.config("2", scale=12)
    lat = B.Sim(w.pos, w.angle, w.hc, w.params).lattice()
    assert lat["active"] and lat["nsub"] == 3 and not lat["inversion_pairs"], lat    # irrational coordinates: T[d] != T[-d] bit for bit
    assert 0 < lat["max_dev"] * 14 < 5e-13 * lat["w_max"]


@pytest.mark.parametrize("geom", ["square_open", "pinwheel_diamond", "ising", "ising_chain"])
def test_stencil_other_geometries(B, geom):
    from oracle import Oracle
    if geom == "square_open":
        pos, ang = W.square_open(37); nd = 2.0
    elif geom == "pinwheel_diamond":
        pos, ang = W.pinwheel_diamond(41); nd = 3.0
    elif geom == "ising":
        pos, ang = W.ising(70, 45); nd = 2.5
    else:
        pos, ang = W.ising(300, 1); nd = 4.0
    N = len(ang)
    p = dict(alpha=0.0013, b=0.4, c=1.0, beta=1.7, gamma=3.0, neighbor_distance=nd)
    hc = W.coercive_fields(N, seed=3)
    spins = W.random_spins(N, seed=9)
    sim = B.Sim(pos, ang, hc, p); sim.set_spins(spins)
    orc = Oracle(pos, ang, hc, p, spins=spins)
    assert sim.lattice()["active"], sim.lattice()
    assert sim.n_interactions == orc.num_interactions and sim.K == orc.build_neighbors()
    for variant in (B.GATHER_STENCIL, B.GATHER_ELL_F64):
        sim.set_gather_variant(variant)
        sim.update_fields()
        assert field_err(sim.get_fields(1).cpu().numpy(), orc.fields(1)) < FIELD_TOL


def test_irregular_geometry_declines_stencil(B):
    """Positions jittered off the lattice: detection must decline and the ELL gather must be exact."""
    from oracle import Oracle
    pos, ang = W.square_closed(20)
    rng = np.random.default_rng(7)
    pos = pos + 0.01 * rng.standard_normal(pos.shape)
    ang = ang + 0.05 * rng.standard_normal(ang.shape)
    N = len(ang)
    p = dict(alpha=0.001, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=1.6)
    hc = W.coercive_fields(N, seed=3); spins = W.random_spins(N, seed=2)
    sim = B.Sim(pos, ang, hc, p); sim.set_spins(spins)
    lat = sim.lattice()
    assert not lat["active"] and lat["reason"] != 0
    with pytest.raises(B.FlatspinError):
        sim.set_gather_variant(B.GATHER_STENCIL)
    orc = Oracle(pos, ang, hc, p, spins=spins)
    sim.update_fields()
    assert field_err(sim.get_fields(1).cpu().numpy(), orc.fields(1)) < FIELD_TOL


def test_partially_jittered_lattice_is_caught_by_verification(B):
    """A lattice whose positions are off by 1e-9 passes the 1e-6 periodicity test but its couplings
    differ at 1e-9: the weight verification must decline the stencil."""
    pos, ang = W.square_closed(16)
    rng = np.random.default_rng(1)
    pos = pos + 1e-9 * rng.standard_normal(pos.shape)
    p = dict(alpha=0.001, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=2.1)   # no shell on the cutoff
    sim = B.Sim(pos, ang, W.coercive_fields(len(ang)), p)
    lat = sim.lattice()
    assert not lat["active"] and lat["reason"] == 8, lat


def test_spin_grid_follows_relax(B):
    """The stencil gather reads dense spin grids that the relax loop keeps in step with its flips: a
    fresh stencil gather after relaxations must equal the oracle's recomputed fields (and the ELL gather)."""
    w = W.config("4", scale=40)
    sim, orc = mk(B, w)
    assert sim.lattice()["active"]
    sim.update_fields()                                   # builds the grids
    for t in (0, 150, 160, 165, 170, 180, 200):
        hx, hy = w.fields[t]
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        assert sim.relax() == orc.relax_B()[0]
        sim.set_gather_variant(B.GATHER_STENCIL); sim.update_fields()
        a = sim.get_fields(1).cpu().numpy()
        assert field_err(a, orc.fields(1)) < FIELD_TOL
        sim.set_gather_variant(B.GATHER_ELL_F64); sim.update_fields()
        assert field_err(sim.get_fields(1).cpu().numpy(), a) < FIELD_TOL
        sim.set_gather_variant(B.GATHER_AUTO)
    assert int((sim.get_spins() == -1).sum()) > 0


def test_stencil_ensemble_matches_ell(B):
    w = W.config("5", scale=30)
    R = 3
    hc = W.coercive_fields(w.N, seed=5, replicas=R)
    sim = B.Sim(w.pos, w.angle, hc, w.params)
    s = np.stack([W.random_spins(w.N, seed=20 + r) for r in range(R)])
    sim.set_spins(s)
    sim.set_gather_variant(B.GATHER_STENCIL); sim.update_fields()
    a = sim.get_fields(1).cpu().numpy()
    sim.set_gather_variant(B.GATHER_ELL_F64); sim.update_fields()
    b = sim.get_fields(1).cpu().numpy()
    assert np.abs(a - b).max() / np.abs(b).max() < 1e-13
    assert not np.array_equal(a[0], a[1])


# ------------------------------------------------------------------ A6/A7: scan
@pytest.mark.parametrize("which,scale", [("1", None), ("3", 20), ("4", 30), ("5", 30)])
def test_scan_candidates_and_argmax(B, which, scale):
    w = W.config(which, scale=scale)
    spins = W.random_spins(w.N, seed=5)
    sim, orc = mk(B, w, spins=spins)
    for t in (0, len(w.fields) // 4, len(w.fields) // 2):
        t = min(t, len(w.fields) - 1)
        hx, hy = w.fields[t]
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        n, best, L = sim.scan()
        no, besto, Lo = orc.scan()
        assert (n, best) == (no, besto)
        if no:
            assert abs(L - Lo) <= 1e-12 * abs(Lo)


# ------------------------------------------------------------------ A7-A9: relaxation, flip order bit-exact
def test_config1_full_protocol_bit_exact(B):
    w = W.config("1")
    total, sim, orc = run_parity(B, w, tier="A", check_fields_every=100)
    assert total == 2 * w.N


def test_config2_kagome_protocol(B):
    w = W.config("2", scale=16)
    total, _, _ = run_parity(B, w, stride=4)
    assert total > w.N


def test_config3_pinwheel_protocol(B):
    w = W.config("3", scale=24)
    total, _, _ = run_parity(B, w, stride=8)
    assert total > w.N // 2


def test_config4_thermal_protocol(B):
    w = W.config("4", scale=60)           # 7320 spins: several leaf blocks and a ragged tail
    total, _, _ = run_parity(B, w, stride=2)
    assert total >= w.N


def test_exact_ties_lowest_index(B):
    pos, ang = W.ising(40, 1)
    p = dict(alpha=0.0, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=1.0)
    sim = B.Sim(pos, ang, np.full(40, 0.1), p)
    sim.set_field(-0.2, 0.05, 0)
    assert sim.relax() == 40
    assert list(sim.get_flip_log().cpu().numpy()) == list(range(40))


def test_max_flips_cap_and_resume(B):
    w = W.config("1")
    sim, orc = mk(B, w)
    hx, hy = w.fields[250]
    sim.set_field(hx, hy, 0); orc.set_field(hx, hy, 0)
    n1 = sim.relax(max_flips=7)
    l1 = sim.get_flip_log().cpu().numpy().copy()
    n2 = sim.relax()
    l2 = sim.get_flip_log().cpu().numpy()
    no, log = orc.relax_B()
    assert n1 == 7 and n1 + n2 == no and np.array_equal(np.concatenate([l1, l2]), log)


def test_run_to_run_determinism(B):
    w = W.config("4", scale=30)
    outs = []
    for _ in range(2):
        sim, _ = mk(B, w)
        logs = []
        for t, (hx, hy) in enumerate(w.fields[::4]):
            sim.set_field(hx, hy, t); sim.relax()
            logs.append(sim.get_flip_log().cpu().numpy().copy())
        outs.append((np.concatenate(logs), sim.get_fields(0).cpu().numpy()))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


# ------------------------------------------------------------------ A10: ensembles
def test_ensemble_matches_independent_oracles(B):
    from oracle import Oracle
    w = W.config("1")
    R = 5
    hc = W.coercive_fields(w.N, seed=100, replicas=R)
    sim = B.Sim(w.pos, w.angle, hc, w.params)
    sim.set_thermal(0.005, 42)
    orcs = [Oracle(w.pos, w.angle, hc[r], w.params, spins=w.spins) for r in range(R)]
    for r, o in enumerate(orcs):
        o.set_thermal(0.005, 42 + r)
    for t, (hx, hy) in enumerate(w.fields[::25]):
        sim.set_field(hx, hy, t)
        n = sim.relax_ensemble()
        for r, o in enumerate(orcs):
            o.set_field(hx, hy, t)
            no, log = o.relax_B()
            assert n[r] == no
            assert np.array_equal(sim.get_flip_log(replica=r).cpu().numpy(), log)
    s = sim.get_spins().cpu().numpy()
    h = sim.get_fields(0).cpu().numpy()
    for r, o in enumerate(orcs):
        assert np.array_equal(s[r], o.spins())
        assert field_err(h[r], o.fields(0)) < FIELD_TOL


# ------------------------------------------------------------------ edge cases / errors
def test_single_spin_and_no_neighbors(B):
    p = dict(alpha=0.001, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=1.0)
    sim = B.Sim(np.array([[0.0, 0.0]]), np.array([0.0]), np.array([0.2]), p)
    assert sim.K == 0 and sim.n_interactions == 0
    sim.set_field(-0.3, 0.0, 0)
    assert sim.relax() == 1 and sim.get_spins().cpu().numpy()[0] == -1
    assert sim.relax() == 0
    # well separated spins: no neighbours at all
    pos = np.stack([np.arange(10) * 5.0, np.zeros(10)], 1)
    sim = B.Sim(pos, np.zeros(10), np.full(10, 0.2), p)
    assert sim.K == 0
    assert np.abs(sim.get_fields(1).cpu().numpy()).max() == 0


def test_errors(B):
    p = dict(alpha=0.001, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=1.0)
    pos = np.array([[0.0, 0.0], [0.0, 0.0]])
    with pytest.raises(B.FlatspinError) as e:
        B.Sim(pos, np.zeros(2), np.full(2, 0.2), p)
    assert e.value.code == B.FS_ERR_COINCIDENT
    with pytest.raises(B.FlatspinError) as e:
        B.Sim(np.array([[0.0, 0.0], [1.0, 0.0]]), np.zeros(2), np.array([0.2, -0.1]), p)
    assert e.value.code == B.FS_ERR_ARG


def test_host_buffer_entry_points(B):
    import torch
    w = W.config("5", scale=20)
    sim, orc = mk(B, w)
    hx, hy = w.fields[0]
    sim.set_field(hx, hy, 0); orc.set_field(hx, hy, 0)
    s_host = torch.as_tensor(w.spins).pin_memory()
    h_host = torch.empty((w.N, 2), dtype=torch.float64).pin_memory()
    n, best, L = sim.step_host(s_host, h_host)
    assert (n, best) == orc.scan()[:2]
    assert field_err(h_host.numpy(), orc.fields(0)) < FIELD_TOL
    assert sim.step_host(s_host, None)[:2] == (n, best)         # summary only: the fields stay on the device
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    w1 = W.config("1")
    sim, orc = mk(B, w1)
    s_out = torch.empty(w1.N, dtype=torch.int8).pin_memory()
    hx, hy = w1.fields[250]
    orc.set_field(hx, hy, 250)
    assert sim.relax_host(hx, hy, 250, s_out) == orc.relax_B()[0]
    assert np.array_equal(s_out.numpy(), orc.spins())


def test_field_by_value_state_machine(B):
    """fs_set_field launches nothing: the value waits for the next scan (kernel argument) or is flushed for the other
    readers.  Every order of calls must see the field that was set last."""
    import torch
    w = W.config("1")
    sim, orc = mk(B, w)

    def ext(sim_):
        return sim_.get_fields(2).cpu().numpy()

    h1, h2, h3 = w.fields[100], w.fields[260], w.fields[300]
    # set -> read the external field before any scan (flush path)
    sim.set_field(*h1, 100); orc.set_field(*h1, 100)
    assert field_err(ext(sim), orc.fields(2)) < FIELD_TOL
    # set twice -> scan sees the second value; the total field afterwards too
    sim.set_field(*h1, 100); sim.set_field(*h2, 260); orc.set_field(*h2, 260)
    assert sim.scan()[:2] == orc.scan()[:2]
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    # set -> relax (scan inside) -> read
    sim.set_field(*h3, 300); orc.set_field(*h3, 300)
    n = sim.relax(); no, log = orc.relax_B()
    assert n == no and np.array_equal(sim.get_flip_log().cpu().numpy(), log)
    assert field_err(ext(sim), orc.fields(2)) < FIELD_TOL
    # a pending value must not survive a sweep (which leaves its own last field) ...
    sim.set_field(*h1, 100)
    fields = w.fields[300:320]
    sim.sweep(fields, step0=300)
    for t, (hx, hy) in enumerate(fields):
        orc.set_field(hx, hy, 300 + t); orc.relax_B()
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(ext(sim), orc.fields(2)) < FIELD_TOL
    assert sim.scan()[:2] == orc.scan()[:2]
    # ... nor an ensemble field upload, nor the host-buffer step
    sim.set_field(*h1, 100)
    sim.set_field_ensemble(np.array([h2]), 260); orc.set_field(*h2, 260)
    assert sim.scan()[:2] == orc.scan()[:2]
    sim.set_field(*h3, 300); orc.set_field(*h3, 300)
    s_host = torch.as_tensor(orc.spins().copy()).pin_memory()
    h_host = torch.empty((w.N, 2), dtype=torch.float64).pin_memory()
    assert sim.step_host(s_host, h_host)[:2] == orc.scan()[:2]
    assert field_err(h_host.numpy(), orc.fields(0)) < FIELD_TOL


@pytest.mark.parametrize("geom,batched", [("square_open", True), ("square_open", False), ("ising", True), ("ising", False)])
def test_other_geometries_whole_protocol(B, geom, batched):
    """Relaxation protocols on the two flatspin geometries no BASELINE config uses: square ASI with
    open edges (the geometry of the paper's own throughput figure: 8-spin neighbourhood) and the 2-D Ising
    lattice (one sublattice, parallel spins), with the thermal field, a generalised astroid and a hysteresis ramp; large
    enough for the batched kernel (>= 16,384 spins), sequential kernel beside it; flip logs against the Tier B oracle."""
    if geom == "square_open":
        pos, ang = W.square_open(92); nd, phi = 1.0, 45.0                # 16,744 spins
        par = dict(alpha=0.001, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=nd)
    else:
        pos, ang = W.ising(130, 130); nd, phi = 1.5, 30.0               # 16,900 spins, 8 neighbours
        par = dict(alpha=0.0008, b=0.41, c=1.0, beta=1.5, gamma=3.9, neighbor_distance=nd)
    N = len(ang)
    w = W.Workload(f"{geom}_protocol", pos, ang, W.coercive_fields(N, seed=5), np.ones(N, np.int8), par,
                   W.ramp(0.22, -0.22, 60, phi, legs=2), sigma_th=0.004, thermal_seed=3)
    sim, orc = mk(B, w)
    assert sim.lattice()["active"]
    if not batched:
        sim.set_batch(0)
    total = 0
    for t, (hx, hy) in enumerate(w.fields):
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        n = sim.relax()
        no, log = orc.relax_B()
        assert n == no, (t, n, no)
        if n:
            assert np.array_equal(sim.get_flip_log().cpu().numpy(), log), t
        total += n
    assert total >= N                                   # at least one full reversal
    if batched:
        assert sim.batch_stats()["flips"] > 0
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    assert orc.monitor()[0] == 0
    sim.update_fields()                                  # a fresh stencil gather of the final state
    assert field_err(sim.get_fields(1).cpu().numpy(), orc.fields(1)) < FIELD_TOL


@pytest.mark.parametrize("n", [15, 24])
def test_cutoff_covers_the_whole_system(B, n):
    """Maximum neighbourhood: the cutoff covers the system, every spin is every other spin's neighbour (K = N - 1: 479
    and 1199, the second more than one pass of the 1024-thread relax kernel); the stencil spans the whole lattice
    (half-extent 15 / 24 cells).  Fields by stencil and by ELL, scan and a whole hysteresis against the oracle."""
    w = W.config("1", scale=n)
    w.params["neighbor_distance"] = 100.0
    w.fields = W.ramp(0.3, -0.3, 40, 45.0, legs=2)
    spins = W.random_spins(w.N, seed=2)
    sim, orc = mk(B, w, spins=spins)
    assert sim.K == w.N - 1 and orc.build_neighbors() == w.N - 1
    lat = sim.lattice()
    assert lat["active"] and lat["Ru"] == n, lat
    hx, hy = w.fields[7]
    sim.set_field(hx, hy, 7); orc.set_field(hx, hy, 7)
    for variant in (B.GATHER_ELL_F64, B.GATHER_STENCIL):
        sim.set_gather_variant(variant); sim.update_fields()
        _check_all_fields(sim, orc)
    assert sim.scan()[:2] == orc.scan()[:2]
    total = 0
    for t, (hx, hy) in enumerate(w.fields):
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        nf = sim.relax(); no, log = orc.relax_B()
        assert nf == no and (nf == 0 or np.array_equal(sim.get_flip_log().cpu().numpy(), log)), t
        total += nf
    assert total > w.N
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL


# ------------------------------------------------------------------ BASELINE.json full sizes
def _full_protocol(B, which, stride=1):
    """Whole protocol of a config at BASELINE.json's full size, Tier B oracle beside the GPU, flip log
    compared step by step.  A mismatch is a failure unless the oracle's near-tie monitor (DESIGN.md W)
    recorded an event (then the input is not well posed and the test reports that instead)."""
    w = W.config(which)
    sim, orc = mk(B, w)
    total = 0
    for t, (hx, hy) in list(enumerate(w.fields))[::stride]:
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        n = sim.relax()
        no, log = orc.relax_B()
        ok = (n == no) and (n == 0 or np.array_equal(sim.get_flip_log().cpu().numpy(), log))
        if not ok:
            ev, gap, thr = orc.monitor()
            assert ev > 0, f"flip sequence differs at step {t} with no near-tie recorded (gap {gap:.2e}, thr {thr:.2e})"
            pytest.xfail(f"near-tie at step {t}: order not well posed (gap {gap:.2e})")
        total += n
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    assert sim.scan()[0] == 0
    return total, w, sim, orc


@pytest.mark.slow
def test_config2_full_size_protocol(B):
    total, w, _, _ = _full_protocol(B, "2")
    assert w.N == 7699 and total > w.N


@pytest.mark.slow
def test_config2b_full_size_protocol(B):
    total, w, _, _ = _full_protocol(B, "2b")
    assert w.N == 14979 and total > w.N


@pytest.mark.slow
def test_config3_full_size_protocol(B):
    total, w, _, _ = _full_protocol(B, "3")                # all 2001 field values
    assert w.N == 80400 and total > w.N


@pytest.mark.slow
def test_config4_full_size_protocol(B):
    total, w, sim, _ = _full_protocol(B, "4")
    assert w.N == 2002000 and total == w.N                  # every spin reverses exactly once (P-8)
    assert bool((sim.get_spins() == -1).all().item())


@pytest.mark.slow
def test_config5_full_size_fields_and_scan(B):
    """Config 5 at full size, in the launch configuration bench.py times (auto = stencil): h_dip and the total field of
    ALL 501,000 spins, from the stencil gather and from the ELL gather, element by element against the oracle's direct
    Eq. 3 evaluation over the 311,247,284 pairs; the scan's switchable count / arg-max against the oracle's full scan."""
    w = W.config("5")
    sim, orc = mk(B, w)
    hx, hy = w.fields[0]
    sim.set_field(hx, hy, 0); orc.set_field(hx, hy, 0)
    assert sim.lattice()["active"] and (sim.N, sim.K, sim.n_interactions) == (501000, 632, 311247284)
    ref_dip, ref_tot = orc.fields(1), orc.fields(0)
    assert ref_dip.shape == (w.N, 2) and np.abs(ref_dip).max() > 0
    sim.update_fields()                                     # auto = the lattice stencil
    assert field_err(sim.get_fields(1).cpu().numpy(), ref_dip) < FIELD_TOL
    assert field_err(sim.get_fields(0).cpu().numpy(), ref_tot) < FIELD_TOL
    sim.set_gather_variant(B.GATHER_ELL_F64); sim.update_fields()
    assert field_err(sim.get_fields(1).cpu().numpy(), ref_dip) < FIELD_TOL
    assert field_err(sim.get_fields(0).cpu().numpy(), ref_tot) < FIELD_TOL
    sim.set_gather_variant(B.GATHER_AUTO); sim.update_fields()
    n, best, L = sim.scan()
    no, besto, Lo = orc.scan()
    assert (n, best) == (no, besto) and abs(L - Lo) <= 1e-12 * abs(Lo)


# ------------------------------------------------------------------ fs_sweep: whole protocol in one launch
@pytest.mark.parametrize("which,scale,stride", [("1", None, 1), ("2", 16, 4), ("3", 24, 8), ("4", 40, 1)])
def test_sweep_one_launch_matches_oracle(B, which, scale, stride):
    w = W.config(which, scale=scale)
    sim, orc = mk(B, w)
    fields = w.fields[::stride]
    steps = list(range(len(w.fields)))[::stride]
    # thermal step keys must equal the protocol's row index: sweep in runs of consecutive keys when strided
    counts, logs = [], []
    for t, (hx, hy) in zip(steps, fields):
        orc.set_field(hx, hy, t)
        n, log = orc.relax_B()
        counts.append(n); logs.append(log)
    if stride == 1:
        n, ps = sim.sweep(fields, step0=0)
        got = ps.cpu().numpy()[0]
        glog = sim.get_flip_log().cpu().numpy()
    else:
        got, glogs = [], []
        for t, f in zip(steps, fields):                   # one-step sweeps keep the step keys of the protocol
            n, ps = sim.sweep(f[None, :], step0=t)
            got.append(int(ps.cpu().numpy()[0, 0])); glogs.append(sim.get_flip_log().cpu().numpy().copy())
        got = np.array(got); glog = np.concatenate(glogs)
    assert np.array_equal(got, np.array(counts))
    ref = np.concatenate(logs) if logs else np.zeros(0, np.int32)
    m = min(len(glog), len(ref))
    assert m > 0 and np.array_equal(glog[:m], ref[:m])
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    assert orc.monitor()[0] == 0


def test_sweep_ensemble(B):
    from oracle import Oracle
    w = W.config("1")
    R = 6
    hc = W.coercive_fields(w.N, seed=300, replicas=R)
    sim = B.Sim(w.pos, w.angle, hc, w.params)
    sim.set_thermal(0.004, 7)
    fields = w.fields[::5]
    n, ps = sim.sweep(fields, step0=0)
    ps = ps.cpu().numpy()
    s = sim.get_spins().cpu().numpy()
    for r in range(R):
        o = Oracle(w.pos, w.angle, hc[r], w.params, spins=w.spins)
        o.set_thermal(0.004, 7 + r)
        cnt, logs = [], []
        for t, (hx, hy) in enumerate(fields):
            o.set_field(hx, hy, t)
            c, log = o.relax_B()
            cnt.append(c); logs.append(log)
        assert np.array_equal(ps[r], np.array(cnt)) and n[r] == sum(cnt)
        assert np.array_equal(sim.get_flip_log(replica=r).cpu().numpy()[: n[r]], np.concatenate(logs)[: 4 * w.N + 1024])
        assert np.array_equal(s[r], o.spins())
    # the per-replica spin grids followed the sweep: a fresh stencil gather equals a fresh ELL gather
    assert sim.lattice()["active"]
    sim.set_gather_variant(B.GATHER_STENCIL); sim.update_fields(); a = sim.get_fields(1).cpu().numpy()
    sim.set_gather_variant(B.GATHER_ELL_F64); sim.update_fields(); b = sim.get_fields(1).cpu().numpy()
    assert np.abs(a - b).max() / np.abs(b).max() < 1e-13


# ------------------------------------------------------------------ per-spin external field
def test_local_field_parity(B):
    """A smooth spatial vector field h_ext(r) sampled per spin, on top of the global ramp: fields, scan, relax
    (stepwise and one-launch sweep) against the oracle; clearing it restores the global-only results."""
    w = W.config("4", scale=30)
    loc = 0.03 * np.stack([np.sin(0.4 * w.pos[:, 0]) * np.cos(0.3 * w.pos[:, 1]),
                           np.cos(0.5 * w.pos[:, 0] + 0.2 * w.pos[:, 1])], axis=1)
    sim, orc = mk(B, w)
    sim.set_local_field(loc); orc.set_local_field(loc)
    hx, hy = w.fields[120]
    sim.set_field(hx, hy, 120); orc.set_field(hx, hy, 120)
    sim.update_fields()
    _check_all_fields(sim, orc)
    assert sim.scan()[:2] == orc.scan()[:2]
    total = 0
    for t in range(120, 200, 4):
        hx, hy = w.fields[t]
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        n = sim.relax(); no, log = orc.relax_B()
        assert n == no and (n == 0 or np.array_equal(sim.get_flip_log().cpu().numpy(), log))
        total += n
    assert total > 0 and np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    # one-launch sweep with the local field, from a fresh state
    sim2, orc2 = mk(B, w)
    sim2.set_local_field(loc); orc2.set_local_field(loc)
    cnt = []
    for t, (hx, hy) in enumerate(w.fields):
        orc2.set_field(hx, hy, t); cnt.append(orc2.relax_B()[0])
    n, ps = sim2.sweep(w.fields, step0=0)
    assert np.array_equal(ps.cpu().numpy()[0], np.array(cnt))
    assert np.array_equal(sim2.get_spins().cpu().numpy(), orc2.spins())
    assert field_err(sim2.get_fields(0).cpu().numpy(), orc2.fields(0)) < FIELD_TOL
    sim2.set_local_field(None); orc2.set_local_field(None)
    assert field_err(sim2.get_fields(2).cpu().numpy(), orc2.fields(2)) < FIELD_TOL


# ------------------------------------------------------------------ more edge cases of the boundary
def test_workspace_errors_and_reuse(B):
    import ctypes as C
    import torch
    L = B.load_library()
    w = W.config("1")
    pos = torch.as_tensor(w.pos).cuda(); ang = torch.as_tensor(w.angle).cuda(); hc = torch.as_tensor(w.hc).cuda()
    p = B.FsParams(*[w.params[k] for k in ("alpha", "b", "c", "beta", "gamma", "neighbor_distance")])
    nbytes = C.c_size_t()
    sp = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    assert L.fs_workspace_bytes(w.N, 1, pos.data_ptr(), C.byref(p), C.byref(nbytes), sp) == 0 and nbytes.value > 0
    ws = torch.empty(nbytes.value + 512, dtype=torch.uint8, device="cuda")
    base = (ws.data_ptr() + 255) // 256 * 256
    h = C.c_void_p()
    # too small, then misaligned: both refused with FS_ERR_WORKSPACE and a message, no handle created
    assert L.fs_create(C.byref(h), w.N, pos.data_ptr(), ang.data_ptr(), hc.data_ptr(), C.byref(p), base, 1024, sp) == B.FS_ERR_WORKSPACE
    assert b"workspace" in L.fs_last_error()
    assert L.fs_create(C.byref(h), w.N, pos.data_ptr(), ang.data_ptr(), hc.data_ptr(), C.byref(p), base + 8, nbytes.value, sp) == B.FS_ERR_WORKSPACE
    # exact size works; the same workspace can be reused after fs_destroy
    for _ in range(2):
        assert L.fs_create(C.byref(h), w.N, pos.data_ptr(), ang.data_ptr(), hc.data_ptr(), C.byref(p), base, nbytes.value, sp) == 0
        n = C.c_int64()
        assert L.fs_set_field(h, -0.2, -0.2, 0) == 0 and L.fs_relax(h, 0, C.byref(n)) == 0 and n.value == w.N
        assert L.fs_destroy(h) == 0
    # null pointers and bad selectors are reported, not dereferenced
    assert L.fs_get_fields(None, 0, None) == B.FS_ERR_ARG
    assert L.fs_sweep(None, None, 3, 0, None, 0, None) == B.FS_ERR_ARG


def test_sweep_max_flips_cap(B):
    w = W.config("1")
    sim, orc = mk(B, w)
    n, ps = sim.sweep(w.fields, step0=0, max_flips=100)
    assert n[0] == 100 and int(ps.sum().item()) == 100          # stopped inside the protocol, state still valid
    ref = []
    for t, (hx, hy) in enumerate(w.fields):
        orc.set_field(hx, hy, t); ref.append(orc.relax_B()[1])
        if sum(len(r) for r in ref) >= 100:
            break
    assert np.array_equal(sim.get_flip_log().cpu().numpy()[:100], np.concatenate(ref)[:100])
    # the state left behind is the one of the step actually reached (t), not of the protocol's last step
    assert int(ps[0, :t].sum().item()) + int(ps[0, t].item()) == 100 and int(ps[0, t + 1:].sum().item()) == 0
    assert field_err(sim.get_fields(2).cpu().numpy(), orc.fields(2)) < FIELD_TOL


def test_many_replicas_more_than_sms(B):
    """R = 300 replicas (> 148 SMs, several CTAs per SM and more than one wave of relax CTAs)."""
    from oracle import Oracle
    pos, ang = W.square_closed(3)
    N = len(ang); R = 300
    p = dict(alpha=0.002, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=1.0)
    hc = W.coercive_fields(N, seed=40, replicas=R)
    sim = B.Sim(pos, ang, hc, p)
    sim.set_field(-0.15, -0.16, 0)
    n = sim.relax_ensemble()
    s = sim.get_spins().cpu().numpy()
    for r in (0, 1, 147, 148, 149, 299):
        o = Oracle(pos, ang, hc[r], p)
        o.set_field(-0.15, -0.16, 0)
        no, log = o.relax_B()
        assert n[r] == no and np.array_equal(sim.get_flip_log(replica=r).cpu().numpy(), log)
        assert np.array_equal(s[r], o.spins())


def test_relax_64_thread_variant_many_replicas(B):
    """R = 1,300 replicas (> 8 per SM): the 64-thread relax CTA (k_relax<64>), the variant bench.py's ensemble
    figure runs.  Stepwise relax and the one-launch sweep, sampled replicas incl. first / last / around 8 x SMs."""
    from oracle import Oracle
    pos, ang = W.square_closed(4)
    N = len(ang); R = 1300
    p = dict(alpha=0.002, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=1.0)
    hc = W.coercive_fields(N, seed=70, replicas=R)
    fields = W.ramp(0.2, -0.2, 40, 45.0, legs=2)
    sample = (0, 1, 147, 148, 1183, 1184, 1185, 1298, 1299)
    # stepwise
    sim = B.Sim(pos, ang, hc, p); sim.set_thermal(0.006, 5)
    orcs = {r: Oracle(pos, ang, hc[r], p) for r in sample}
    for r, o in orcs.items():
        o.set_thermal(0.006, 5 + r)
    tot = 0
    for t, (hx, hy) in enumerate(fields):
        sim.set_field(hx, hy, t)
        n = sim.relax_ensemble()
        for r, o in orcs.items():
            o.set_field(hx, hy, t)
            no, log = o.relax_B()
            assert n[r] == no, (t, r)
            assert np.array_equal(sim.get_flip_log(replica=r).cpu().numpy(), log), (t, r)
            tot += no
    assert tot > len(sample) * N
    s = sim.get_spins().cpu().numpy(); h = sim.get_fields(0).cpu().numpy()
    for r, o in orcs.items():
        assert np.array_equal(s[r], o.spins()) and field_err(h[r], o.fields(0)) < FIELD_TOL
    # one launch
    sim = B.Sim(pos, ang, hc, p); sim.set_thermal(0.006, 5)
    n, ps = sim.sweep(fields, step0=0)
    ps = ps.cpu().numpy(); s = sim.get_spins().cpu().numpy()
    for r in sample:
        o = Oracle(pos, ang, hc[r], p); o.set_thermal(0.006, 5 + r)
        cnt, logs = [], []
        for t, (hx, hy) in enumerate(fields):
            o.set_field(hx, hy, t); c, log = o.relax_B(); cnt.append(c); logs.append(log)
        assert np.array_equal(ps[r], np.array(cnt)) and n[r] == sum(cnt)
        assert np.array_equal(sim.get_flip_log(replica=r).cpu().numpy()[: n[r]], np.concatenate(logs))
        assert np.array_equal(s[r], o.spins())


def test_stencil_shared_memory_table_variant(B):
    """A coupling table too large for the 56 KB constant bank (square ASI, neighbor distance 15: 4 x 31 x 31 =
    3,844 entries): k_gather_stencil reads the table from shared memory instead.  Fields against the oracle."""
    from oracle import Oracle
    pos, ang = W.square_closed(40)
    N = len(ang)
    p = dict(alpha=0.001, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=15.0)
    hc = W.coercive_fields(N, seed=3); spins = W.random_spins(N, seed=12)
    sim = B.Sim(pos, ang, hc, p); sim.set_spins(spins)
    lat = sim.lattice()
    assert lat["active"] and (lat["Ru"], lat["Rv"]) == (15, 15) and lat["nsub"] ** 2 * 31 * 31 > 3584, lat
    orc = Oracle(pos, ang, hc, p, spins=spins)
    sim.set_gather_variant(B.GATHER_STENCIL); sim.update_fields()
    a = sim.get_fields(1).cpu().numpy()
    assert field_err(a, orc.fields(1)) < FIELD_TOL
    sim.set_gather_variant(B.GATHER_ELL_F64); sim.update_fields()
    assert field_err(sim.get_fields(1).cpu().numpy(), a) < FIELD_TOL


def test_two_sims_of_different_size_stay_usable(B):
    """The dynamic shared-memory limit of a kernel belongs to the function, not to a simulation: creating a
    small simulation after a large one must not break the large one's relax / stencil gather."""
    w3 = W.config("4", scale=200)                     # 80,400 spins: ~100 KB of relax shared memory (leaf hierarchy)
    simA, orcA = mk(B, w3)
    w1 = W.config("1")
    simB, orcB = mk(B, w1)                            # created afterwards, far smaller
    hx, hy = w3.fields[160]
    simA.set_field(hx, hy, 160); orcA.set_field(hx, hy, 160)
    n = simA.relax(); no, log = orcA.relax_B()
    assert n == no and n > 0 and np.array_equal(simA.get_flip_log().cpu().numpy(), log)
    simA.set_gather_variant(B.GATHER_STENCIL); simA.update_fields()
    assert field_err(simA.get_fields(1).cpu().numpy(), orcA.fields(1)) < FIELD_TOL
    hx, hy = w1.fields[250]
    simB.set_field(hx, hy, 250); orcB.set_field(hx, hy, 250)
    assert simB.relax() == orcB.relax_B()[0]


def test_annealing_sweep_matches_oracle(B):
    """annealing = a protocol whose thermal field strength decreases exponentially.  One launch
    (fs_sweep_anneal) against the oracle stepping the same sigma_t, on the 50x50-style recipe of PAPER.md:196
    scaled down (square closed, b = 0.4, nd = 3), zero external field."""
    pos, ang = W.square_closed(14)
    N = len(ang)
    p = dict(alpha=0.0018, b=0.4, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=3.0)
    hc = W.coercive_fields(N, hk=0.186, seed=9)
    spins = W.random_spins(N, seed=4)
    from oracle import Oracle
    sim = B.Sim(pos, ang, hc, p); sim.set_spins(spins); sim.set_thermal(0.0, 77)
    orc = Oracle(pos, ang, hc, p, spins=spins)
    T = 60
    sigma = 0.12 * np.exp(-np.arange(T) / 12.0)
    fields = np.zeros((T, 2))
    cnt = []
    for t in range(T):
        orc.set_thermal(float(sigma[t]), 77); orc.set_field(0.0, 0.0, t)
        cnt.append(orc.relax_B()[0])
    n, ps = sim.sweep(fields, step0=0, sigma=sigma)
    assert sum(cnt) > 50 and np.array_equal(ps.cpu().numpy()[0], np.array(cnt))
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    sim.set_thermal(float(sigma[-1]), 77)
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    assert orc.monitor()[0] == 0


@pytest.mark.parametrize("which,scale,stride", [("4", 120, 1), ("3", 50, 4), ("2", 30, 2), ("1", 24, 1)])
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_other_disorder_and_thermal_seeds(B, which, scale, stride, seed):
    """Bit-exact flip sequences are not luck of seed 0: other h_c disorder draws and thermal seeds."""
    from oracle import Oracle
    w = W.config(which, scale=scale)
    hc = W.coercive_fields(w.N, seed=seed)
    sim = B.Sim(w.pos, w.angle, hc, w.params); orc = Oracle(w.pos, w.angle, hc, w.params, spins=w.spins)
    sim.set_spins(w.spins)
    if w.sigma_th:
        sim.set_thermal(w.sigma_th, seed + 10); orc.set_thermal(w.sigma_th, seed + 10)
    total = 0
    for t, (hx, hy) in list(enumerate(w.fields))[::stride]:
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        n = sim.relax(); no, log = orc.relax_B()
        if n != no or (n and not np.array_equal(sim.get_flip_log().cpu().numpy(), log)):
            ev, gap, thr = orc.monitor()
            assert ev > 0, f"flip sequence differs at step {t} with no near-tie recorded"
            pytest.xfail(f"near-tie at step {t} (gap {gap:.1e}): order not well posed")
        total += n
    assert total >= w.N
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL


# ------------------------------------------------------------------ the paper's own parameter sets as workloads
def test_paper_pinwheel_reversal_parameters(B):
    """PAPER.md:230 (IV.C): 25x25 pinwheel diamond = 1250 magnets, nd = 10, beta = 4.8 (general
    exponent path), field at 30 degrees: two-step reversal.  Every 25th of the 2501 field values."""
    w = W.paper_pinwheel_reversal(25, 30.0)
    assert w.N == 1250
    total, sim, orc = run_parity(B, w, stride=25)
    assert total >= w.N and sim.K == 632


def test_paper_kagome_dirac_string_parameters(B):
    """PAPER.md:180-182 (IV.A): 29x29 hexagons = 2638 magnets, beta = 2.5, b = 0.212, sigma_th = 0.002."""
    w = W.paper_kagome_dirac_strings(29, K=200)
    assert w.N == 2638
    total, sim, orc = run_parity(B, w, stride=2)
    assert total > w.N // 4


# ------------------------------------------------------------------ f1: exact batched flips (k_relax_batch)
def _protocol_vs_oracle(B, w, steps, hc=None, expect_batched=True):
    """Relax at the given protocol steps with the batched kernel active; flip logs against the Tier B oracle."""
    from oracle import Oracle
    hc = w.hc if hc is None else hc
    sim = B.Sim(w.pos, w.angle, hc, w.params); sim.set_spins(w.spins)
    orc = Oracle(w.pos, w.angle, hc, w.params, spins=w.spins)
    if w.sigma_th:
        sim.set_thermal(w.sigma_th, w.thermal_seed); orc.set_thermal(w.sigma_th, w.thermal_seed)
    assert sim.batch_stats()["max_seeds"] > 0, "batched flips should be available for this size"
    total = 0
    for t in steps:
        hx, hy = w.fields[t]
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        n = sim.relax(); no, log = orc.relax_B()
        assert n == no, (t, n, no)
        if n:
            assert np.array_equal(sim.get_flip_log().cpu().numpy(), log), f"flip order differs at step {t}"
        total += n
    st = sim.batch_stats()
    if expect_batched:
        assert st["flips"] > total // 2 and st["rounds"] > 0, st      # the batched kernel did most of the work
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    assert field_err(sim.get_fields(1).cpu().numpy(), orc.fields(1)) < FIELD_TOL     # incremental h_dip incl. undone rounds
    assert orc.monitor()[0] == 0 and sim.scan()[0] == 0
    return total, st, sim


def test_batched_flips_config4_bit_exact(B):
    w = W.config("4", scale=120)                       # 29,040 spins, thermal ramp: every spin reverses
    total, st, sim = _protocol_vs_oracle(B, w, range(len(w.fields)))
    assert total == w.N
    # the stencil spin grid followed the committed flips only (undone ones never reach it)
    sim.set_gather_variant(B.GATHER_STENCIL); sim.update_fields(); a = sim.get_fields(1).cpu().numpy()
    sim.set_gather_variant(B.GATHER_ELL_F64); sim.update_fields(); b = sim.get_fields(1).cpu().numpy()
    assert field_err(a, b) < 1e-13


def test_batched_flips_one_giant_avalanche_refines_threshold(B):
    """A single field jump makes every spin switchable at once with margins inside a few histogram bins: the
    threshold search must split a bin (linear refinement pass) and the whole array reverses in one relax."""
    w = W.config("4", scale=100)                       # 20,200 spins
    w.fields = np.array([[-0.25 * math.cos(math.pi / 4), -0.25 * math.sin(math.pi / 4)]])
    total, st, _ = _protocol_vs_oracle(B, w, [0], expect_batched=False)   # (it hands over to k_relax once rounds run lean)
    assert total == w.N and st["rounds"] > 10 and st["flips"] > 1000


@pytest.mark.parametrize("which,scale,stride", [("3", 100, 4), ("2", 80, 2)])
def test_batched_flips_other_lattices(B, which, scale, stride):
    """K = 60 (two chunks of neighbours per flip, domino avalanches: the kernel hands over to k_relax when its
    prefixes stay short) and the kagome lattice (K = 14, three sublattices)."""
    w = W.config(which, scale=scale)
    assert w.N >= 16384
    total, st, _ = _protocol_vs_oracle(B, w, range(0, len(w.fields), stride), expect_batched=False)
    assert total > w.N // 2


def test_batched_equals_sequential_with_exact_ties(B):
    """Uniform h_c and a symmetric start: whole classes of spins have bit-identical margins, so the order among
    them is decided by the index alone.  The batched kernel (threshold search over identical keys, bail-out when a
    single key value exceeds the round's capacity) must give the sequential kernel's log bit for bit."""
    pos, ang = W.square_closed(100)
    N = len(ang)
    p = dict(alpha=0.001, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=1.0)
    hc = np.full(N, 0.2)
    fields = W.ramp(0.0, -0.25, 25, 45.0, legs=1)
    logs = {}
    for mode in ("batch", "seq"):
        sim = B.Sim(pos, ang, hc, p)
        if mode == "seq":
            sim.set_batch(0)
        out = []
        for t, (hx, hy) in enumerate(fields):
            sim.set_field(hx, hy, t)
            if sim.relax():
                out.append(sim.get_flip_log().cpu().numpy().copy())
        logs[mode] = (np.concatenate(out), sim.get_spins().cpu().numpy(), sim.get_fields(0).cpu().numpy())
    assert len(logs["seq"][0]) == N
    assert np.array_equal(logs["batch"][0], logs["seq"][0])
    assert np.array_equal(logs["batch"][1], logs["seq"][1]) and np.array_equal(logs["batch"][2], logs["seq"][2])
    # no coupling at all: every spin of a sublattice ties exactly; lowest index first (reading C-7)
    pos, ang = W.ising(20000, 1)
    sim = B.Sim(pos, ang, np.full(20000, 0.1), dict(p, alpha=0.0))
    assert sim.batch_stats()["max_seeds"] > 0
    sim.set_field(-0.2, 0.05, 0)
    assert sim.relax() == 20000
    assert np.array_equal(sim.get_flip_log().cpu().numpy(), np.arange(20000))


@pytest.mark.slow
def test_batched_equals_sequential_config4_full_size(B):
    """2,002,000 spins: batched against the one-flip-at-a-time kernel (which the oracle checks in
    test_config4_full_size_protocol), whole protocol, log of every step."""
    w = W.config("4")
    logs = {}
    for mode in ("batch", "seq"):
        sim = B.Sim(w.pos, w.angle, w.hc, w.params); sim.set_thermal(w.sigma_th, w.thermal_seed)
        if mode == "seq":
            sim.set_batch(0)
        out = []
        for t, (hx, hy) in enumerate(w.fields):
            sim.set_field(hx, hy, t)
            if sim.relax():
                out.append(sim.get_flip_log().cpu().numpy().copy())
        logs[mode] = (np.concatenate(out), sim.get_fields(1).cpu().numpy(), sim.batch_stats())
        sim.close()
    assert np.array_equal(logs["batch"][0], logs["seq"][0]) and np.array_equal(logs["batch"][1], logs["seq"][1])
    st = logs["batch"][2]
    assert st["flips"] > 1_900_000 and st["flips"] / st["rounds"] > 100, st


# ------------------------------------------------------------------ f2: time-dependent protocols, local field series
def _oracle_protocol(orc, fields, local=None):
    counts, logs = [], []
    for t, (hx, hy) in enumerate(fields):
        if local is not None:
            orc.set_local_field(local[t])
        orc.set_field(hx, hy, t)
        n, log = orc.relax_B()
        counts.append(n); logs.append(log)
    return np.array(counts), (np.concatenate(logs) if logs else np.zeros(0, np.int32))


@pytest.mark.parametrize("kind", ["rotating", "sinusoidal", "sawtooth"])
def test_periodic_field_protocols_one_launch(B, kind):
    """Input encoders of PAPER.md:63 / :156: spins flip back and forth over several periods.  One launch (fs_sweep)
    and the stepwise path against the Tier B oracle; a run that makes more flips than the ring log holds must
    return the LAST 4N+1024 flips."""
    from oracle import Oracle
    pos, ang = W.square_closed(16)
    N = len(ang)
    p = dict(alpha=0.001, b=0.4, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=1.5)
    hc = W.coercive_fields(N, seed=8)
    if kind == "rotating":
        fields = W.rotating(0.13, 5, 48, 20.0)
    elif kind == "sinusoidal":
        fields = W.sinusoidal(0.16, 3, 40, 35.0)
    else:
        fields = W.sawtooth(0.16, 3, 40, 35.0)
    orc = Oracle(pos, ang, hc, p)
    counts, ref = _oracle_protocol(orc, fields)
    assert counts.sum() > 2 * N and orc.monitor()[0] == 0            # every spin reverses more than once
    sim = B.Sim(pos, ang, hc, p)
    n, ps = sim.sweep(fields, step0=0)
    assert np.array_equal(ps.cpu().numpy()[0], counts) and n[0] == counts.sum()
    cap = 4 * N + 1024
    glog = sim.get_flip_log().cpu().numpy()
    if counts.sum() > cap:
        assert sim.last_log_first == counts.sum() - cap and len(glog) == cap
        assert np.array_equal(glog, ref[-cap:])
        small = sim.get_flip_log(cap=100).cpu().numpy()             # a short buffer gets the oldest retained flips
        assert np.array_equal(small, ref[-cap:][:100])
    else:
        assert sim.last_log_first == 0 and np.array_equal(glog, ref)
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    # stepwise
    sim2 = B.Sim(pos, ang, hc, p)
    got = []
    for t, (hx, hy) in enumerate(fields):
        sim2.set_field(hx, hy, t); got.append(sim2.relax())
    assert np.array_equal(np.array(got), counts)
    assert np.array_equal(sim2.get_spins().cpu().numpy(), orc.spins())


def test_sweep_local_scale_and_series(B):
    """h_ext^(i)(t) = global(t) + scale(t) * local_i + series(t, i): one launch against the oracle
    stepping the same per-spin field (composed on the host in the same order of operations)."""
    from oracle import Oracle
    w = W.config("4", scale=16)
    T = 60
    fields = W.ramp(0.05, -0.12, T - 1, 45.0)
    loc = 0.04 * np.stack([np.sin(0.5 * w.pos[:, 0]), np.cos(0.4 * w.pos[:, 1])], axis=1)
    scale = np.linspace(0.0, 1.5, T)
    rng = np.random.default_rng(5)
    series = 0.01 * rng.standard_normal((T, w.N, 2))
    cases = {"scale": (loc, scale, None), "series": (None, None, series), "both": (loc, scale, series), "static": (loc, None, None)}
    for name, (l, sc, ser) in cases.items():
        local = []
        for t in range(T):
            tot = np.zeros((w.N, 2))
            if l is not None:
                tot = (sc[t] * l) if sc is not None else l.copy()
            if ser is not None:
                tot = (tot + ser[t]) if l is not None else ser[t].copy()
            local.append(tot)
        orc = Oracle(w.pos, w.angle, w.hc, w.params); orc.set_thermal(w.sigma_th, 3)
        counts, ref = _oracle_protocol(orc, fields, local)
        sim = B.Sim(w.pos, w.angle, w.hc, w.params); sim.set_thermal(w.sigma_th, 3)
        if l is not None:
            sim.set_local_field(l)
        n, ps = sim.sweep(fields, step0=0, local_scale=sc, local_series=ser)
        assert np.array_equal(ps.cpu().numpy()[0], counts), name
        assert counts.sum() > w.N // 4 and np.array_equal(sim.get_flip_log().cpu().numpy(), ref), name
        assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins()), name


# ------------------------------------------------------------------ f4: analysis reductions, the IV.B annealing workload
@pytest.mark.parametrize("geom", ["square_nd3", "rotated_nd2", "kagome"])
def test_spin_correlation_matches_oracle(B, geom):
    from oracle import Oracle
    if geom == "square_nd3":
        pos, ang = W.square_closed(13); nd = 3.0
    elif geom == "rotated_nd2":
        pos, ang = W.rotated_square(11); nd = 2.0
    else:
        pos, ang = W.kagome(9); nd = 2.0
    N = len(ang)
    p = dict(alpha=0.001, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=nd)
    R = 3
    hc = W.coercive_fields(N, seed=2, replicas=R)
    spins = np.stack([W.random_spins(N, seed=30 + r) for r in range(R)])
    sim = B.Sim(pos, ang, hc, p); sim.set_spins(spins)
    for width, nbins in ((0.25, 16), (0.4, 5), (1.0, 3)):
        sm, cnt = sim.correlation(width, nbins)
        sm = sm.cpu().numpy(); cnt = cnt.cpu().numpy()
        for r in range(R):
            o = Oracle(pos, ang, hc[r], p, spins=spins[r])
            osm, ocnt = o.spin_correlation(width, nbins)
            assert np.array_equal(sm[r], osm) and np.array_equal(cnt, ocnt), (geom, width, r)
        assert cnt.sum() > 0


def test_vertex_populations_match_oracle(B):
    from oracle import Oracle
    n = 14
    pos, ang = W.square_closed(n)
    N = len(ang); V = W.square_vertices(n)
    p = dict(alpha=0.001, b=1.0, c=1.0, beta=3.0, gamma=3.0, neighbor_distance=1.0)
    states = [np.ones(N, np.int8), W.square_ground_state(n), W.random_spins(N, seed=1), W.random_spins(N, seed=2)]
    g = W.square_ground_state(n).copy(); g[V[5][1]] *= -1; states.append(g)
    hc = np.full((len(states), N), 0.2)
    sim = B.Sim(pos, ang, hc, p); sim.set_spins(np.stack(states))
    got = sim.vertex_populations(V).cpu().numpy()
    for r, s in enumerate(states):
        o = Oracle(pos, ang, hc[r], p, spins=s)
        assert list(got[r]) == list(o.vertex_populations(V)), r
    assert list(got[0]) == [0, (n - 1) ** 2, 0, 0] and list(got[1]) == [(n - 1) ** 2, 0, 0, 0]
    assert list(got[4]) == [(n - 1) ** 2 - 2, 0, 2, 0] and got[2].sum() == (n - 1) ** 2
    # pinwheel: the same vertices of the rotated lattice
    pos, ang = W.rotated_square(n)
    s = W.random_spins(N, seed=7)
    sim = B.Sim(pos, ang, np.full(N, 0.2), p); sim.set_spins(s)
    o = Oracle(pos, ang, np.full(N, 0.2), p, spins=s)
    assert list(sim.vertex_populations(V).cpu().numpy()) == list(o.vertex_populations(V))


def test_paper_square_anneal_ensemble(B):
    """PAPER.md:196-206 (IV.B) scaled down: an ensemble of square ASIs annealed by an exponentially decreasing thermal
    field in one launch; annealed spins, spin-spin correlation and vertex populations of every replica against
    independent oracles."""
    from oracle import Oracle
    R = 4
    w = W.paper_square_anneal(12, alpha=0.004, T=50, sigma0=0.12, decay=10.0, replicas=R)
    w.params["neighbor_distance"] = 3.0
    sigma, V = w.extra["sigma"], w.extra["vertices"]
    sim = B.Sim(w.pos, w.angle, w.hc, w.params)
    sim.set_spins(np.tile(w.spins, (R, 1))); sim.set_thermal(0.0, 11)
    n, _ = sim.sweep(w.fields, step0=0, sigma=sigma)
    s = sim.get_spins().cpu().numpy()
    sm, cnt = sim.correlation(0.5, 8); sm = sm.cpu().numpy(); cnt = cnt.cpu().numpy()
    vp = sim.vertex_populations(V).cpu().numpy()
    total = 0
    for r in range(R):
        o = Oracle(w.pos, w.angle, w.hc[r], w.params, spins=w.spins)
        for t in range(len(sigma)):
            o.set_thermal(float(sigma[t]), 11 + r); o.set_field(0.0, 0.0, t)
            total += o.relax_B()[0]
        assert np.array_equal(s[r], o.spins()), r
        osm, ocnt = o.spin_correlation(0.5, 8)
        assert np.array_equal(sm[r], osm) and np.array_equal(cnt, ocnt)
        assert list(vp[r]) == list(o.vertex_populations(V))
        assert o.monitor()[0] == 0
    assert total == int(n.sum()) and total > R * w.N // 2
    # annealing lowers the dipolar energy: more minimised nearest-neighbour pairs than in the random start
    o0 = Oracle(w.pos, w.angle, w.hc[0], w.params, spins=w.spins)
    assert sm[0][1] > o0.spin_correlation(0.5, 8)[0][1]


@pytest.mark.parametrize("R", [200, 1300])
def test_many_replicas_with_more_than_31_neighbors(B, R):
    """Ensembles whose update does not fit one warp (K + 1 > 32) and with more replicas than SMs: 256-thread CTAs
    (four replicas per SM), 128-thread ones from eight replicas per SM; a sample of the replicas against independent
    oracles, whole protocol in one launch and stepwise."""
    from oracle import Oracle
    w = W.config("3", scale=6)                              # pinwheel recipe, neighbor distance 3: K = 60 > 31
    hc = W.coercive_fields(w.N, seed=77, replicas=R)
    sim = B.Sim(w.pos, w.angle, hc, w.params)
    assert sim.K + 1 > 32
    fields = w.fields[::40]
    sim.set_spins(np.ones((R, w.N), np.int8))
    n, per = sim.sweep(fields, step0=0)
    s = sim.get_spins().cpu().numpy(); per = per.cpu().numpy()
    sample = sorted({0, 1, R // 2, R - 2, R - 1})
    for r in sample:
        o = Oracle(w.pos, w.angle, hc[r], w.params, spins=np.ones(w.N, np.int8))
        cnt, logs = [], []
        for t, (hx, hy) in enumerate(fields):
            o.set_field(hx, hy, t)
            c, log = o.relax_B()
            cnt.append(c); logs.append(log)
        assert np.array_equal(s[r], o.spins()), r
        assert list(per[r]) == cnt and int(n[r]) == sum(cnt), r
        assert np.array_equal(sim.get_flip_log(replica=r).cpu().numpy()[: int(n[r])], np.concatenate(logs)[: 4 * w.N + 1024]), r
    assert int(n.sum()) > 0
    # stepwise (fs_set_field_ensemble + fs_relax_ensemble) from the same start
    sim.set_spins(np.ones((R, w.N), np.int8)); sim.update_fields()
    for t, (hx, hy) in enumerate(fields):
        sim.set_field(hx, hy, t); sim.relax_ensemble()
    assert np.array_equal(sim.get_spins().cpu().numpy(), s)


def test_more_than_8192_leaves(B):
    """8.8 M spins: 1024-spin leaves, 8,618 of them (the hierarchy's shared memory holds up to 16,384: 16.7 M spins).
    Config-4 recipe at 2100 x 2100 with the thermal field, a few field values around the onset of the reversal, sequential
    and batched relax against the Tier B oracle."""
    w = W.config("4", scale=2100)
    assert w.N > 8192 * 1024
    for batched in (True, False):
        sim, orc = mk(B, w)
        if not batched:
            sim.set_batch(0)
        total = 0
        for t in (0, 120, 128, 131, 134):
            hx, hy = w.fields[t]
            sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
            n = sim.relax()
            no, log = orc.relax_B()
            assert n == no, (t, n, no)
            if n:
                assert np.array_equal(sim.get_flip_log().cpu().numpy(), log[: 4 * w.N + 1024]), t
            total += n
        assert total > 100
        assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
        assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
        assert sim.scan()[0] == orc.scan()[0]
        sim.close(); del orc


# ------------------------------------------------------------------ optional fp32 field path (reported separately, 1e-5)
@pytest.mark.parametrize("which,scale", [("1", None), ("3", 30), ("5", 40), ("2", 20)])
def test_fp32_stencil_field_path(B, which, scale):
    """BASELINE.json north_star: "an optional fp32 field path is reported separately at 1e-5".  The single-precision
    stencil gather against the oracle's fp64 fields, relative to max|h|; it is never the automatic choice and no
    flip-order claim is attached to it.  Kagome (no inversion pairing) exercises the unpaired fp32 kernel."""
    w = W.config(which, scale=scale)
    spins = W.random_spins(w.N, seed=21)
    sim, orc = mk(B, w, spins=spins)
    assert sim.lattice()["active"]
    sim.set_gather_variant(B.GATHER_STENCIL_F32); sim.update_fields()
    a = sim.get_fields(1).cpu().numpy()
    ref = orc.fields(1)
    err = field_err(a, ref)
    assert 0 < err < 1e-5, err                          # single precision: not bit-equal to the fp64 path, well inside the bar
    sim.set_gather_variant(B.GATHER_AUTO); sim.update_fields()
    assert field_err(sim.get_fields(1).cpu().numpy(), ref) < FIELD_TOL        # and the fp64 table is back in place
    # an irregular geometry has no fp32 path
    pos = w.pos + 0.01 * np.random.default_rng(1).standard_normal(w.pos.shape)
    sim2 = B.Sim(pos, w.angle, w.hc, w.params)
    with pytest.raises(B.FlatspinError):
        sim2.set_gather_variant(B.GATHER_STENCIL_F32)


# ------------------------------------------------------------------ geometries that are NOT lattices: the general path
# north_star (a): "a neighbor-list / cell-grid builder, plus a per-sublattice stencil for regular lattices".  Everything
# above runs on detected lattices; these run the other half of the product against the oracle: ragged ELL rows,
# GATHER_AUTO -> ELL, scan, k_relax and k_relax_batch without the lattice's cell index, fs_sweep, ensembles.
OFF_LATTICE = [("jittered_square", 100), ("point_cloud", 20000)]


@pytest.mark.parametrize("kind,n", OFF_LATTICE)
def test_off_lattice_tables_fields_and_scan(B, kind, n):
    w = W.off_lattice(kind, n, seed=1)
    spins = W.random_spins(w.N, seed=4)
    sim, orc = mk(B, w, spins=spins)
    lat = sim.lattice()
    assert not lat["active"] and lat["reason"] != 0, lat
    with pytest.raises(B.FlatspinError):
        sim.set_gather_variant(B.GATHER_STENCIL)
    ref = orc.neighbors()
    assert sim.K == ref.shape[1] and sim.n_interactions == orc.num_interactions
    assert np.array_equal(sim.get_neighbors().cpu().numpy(), ref)
    deg = (ref >= 0).sum(1)
    assert deg.min() < deg.max() == sim.K                   # ragged rows
    for t in (0, len(w.fields) // 2, len(w.fields) - 1):
        hx, hy = w.fields[t]
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        sim.update_fields()
        _check_all_fields(sim, orc)                         # total, dipolar, external, thermal
        ng, best, L = sim.scan()
        no, besto, Lo = orc.scan()
        assert (ng, best) == (no, besto)
        if no:
            assert abs(L - Lo) <= 1e-12 * abs(Lo)


def _off_lattice_protocol(B, w, batched):
    sim, orc = mk(B, w)
    assert not sim.lattice()["active"]
    if batched:
        assert sim.batch_stats()["max_seeds"] > 0, "batched flips should be available for this size"
    else:
        sim.set_batch(0)
    total = 0
    for t, (hx, hy) in enumerate(w.fields):
        sim.set_field(hx, hy, t); orc.set_field(hx, hy, t)
        n = sim.relax(); no, log = orc.relax_B()
        assert n == no, (t, n, no)
        if n:
            assert np.array_equal(sim.get_flip_log().cpu().numpy(), log), f"flip order differs at step {t}"
        total += n
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    assert field_err(sim.get_fields(1).cpu().numpy(), orc.fields(1)) < FIELD_TOL     # incrementally maintained h_dip
    assert orc.monitor()[0] == 0 and sim.scan()[0] == 0
    return total, sim.batch_stats()


@pytest.mark.parametrize("batched", [True, False])
@pytest.mark.parametrize("kind,n", OFF_LATTICE)
def test_off_lattice_whole_protocol(B, kind, n, batched):
    """Thermal ramp 0.2 -> -0.2 on >= 20,000 magnets off any lattice: flip logs of k_relax_batch + k_relax, and of
    k_relax alone, against Tier B, every field value."""
    w = W.off_lattice(kind, n, seed=2)
    assert w.N >= 16384
    total, st = _off_lattice_protocol(B, w, batched)
    assert total > w.N // 2
    if batched:
        assert st["flips"] > 0 and st["rounds"] > 0, st
    else:
        assert st["max_seeds"] == 0 and st["flips"] == 0, st


@pytest.mark.parametrize("kind,n", [("jittered_square", 30), ("point_cloud", 2000)])
def test_off_lattice_sweep_one_launch(B, kind, n):
    w = W.off_lattice(kind, n, seed=3)
    sim, orc = mk(B, w)
    assert not sim.lattice()["active"]
    counts, logs = [], []
    for t, (hx, hy) in enumerate(w.fields):
        orc.set_field(hx, hy, t)
        c, log = orc.relax_B()
        counts.append(c); logs.append(log)
    nf, ps = sim.sweep(w.fields, step0=0)
    assert np.array_equal(ps.cpu().numpy()[0], np.array(counts)) and int(nf[0]) == sum(counts)
    assert np.array_equal(sim.get_flip_log().cpu().numpy(), np.concatenate(logs))
    assert sum(counts) > w.N // 2
    assert np.array_equal(sim.get_spins().cpu().numpy(), orc.spins())
    assert field_err(sim.get_fields(0).cpu().numpy(), orc.fields(0)) < FIELD_TOL
    assert orc.monitor()[0] == 0


def test_off_lattice_ensemble(B):
    from oracle import Oracle
    w = W.off_lattice("point_cloud", 1500, seed=5)
    R = 4
    hc = W.coercive_fields(w.N, seed=200, replicas=R)
    sim = B.Sim(w.pos, w.angle, hc, w.params)
    assert not sim.lattice()["active"]
    sim.set_thermal(w.sigma_th, 42)
    orcs = [Oracle(w.pos, w.angle, hc[r], w.params, spins=w.spins) for r in range(R)]
    for r, o in enumerate(orcs):
        o.set_thermal(w.sigma_th, 42 + r)
    flips = 0
    for t, (hx, hy) in enumerate(w.fields):
        sim.set_field(hx, hy, t)
        n = sim.relax_ensemble()
        for r, o in enumerate(orcs):
            o.set_field(hx, hy, t)
            no, log = o.relax_B()
            assert n[r] == no
            assert np.array_equal(sim.get_flip_log(replica=r).cpu().numpy()[:no], log)
            flips += no
    assert flips > R * w.N // 2
    s = sim.get_spins().cpu().numpy(); h = sim.get_fields(0).cpu().numpy()
    for r, o in enumerate(orcs):
        assert np.array_equal(s[r], o.spins())
        assert field_err(h[r], o.fields(0)) < FIELD_TOL
        assert o.monitor()[0] == 0


# ------------------------------------------------------------------ boundary: device memory comes from the caller
def test_device_memory_is_the_callers_workspace(B):
    """the workspace is caller-allocated.  Driver free memory + torch's reserved pool stays constant unless
    somebody other than torch allocates, so its drop across fs_create is exactly what the library allocated itself:
    nothing for a geometry that is not a lattice, the stencil table set (bounded by 8N + 2^20 cells per grid) for a
    lattice -- and nothing more during set_local_field, batched relaxation, sweeps or reads."""
    import torch

    def outside_torch():
        torch.cuda.synchronize()
        return torch.cuda.mem_get_info()[0] + torch.cuda.memory_reserved()

    for make, lattice in ((lambda: W.off_lattice("point_cloud", 20000, seed=6), False), (lambda: W.config("4", scale=110), True)):
        w = make()
        for attempt in range(2):                            # the first pass loads the kernels (module memory), the second is measured
            base = outside_torch()
            sim = B.Sim(w.pos, w.angle, w.hc, w.params)
            owned = base - outside_torch()
            assert sim.lattice()["active"] == lattice and sim.batch_stats()["max_seeds"] > 0
            sim.set_spins(w.spins); sim.set_thermal(w.sigma_th, w.thermal_seed)
            rng = np.random.default_rng(0)
            sim.set_local_field(1e-3 * rng.standard_normal((w.N, 2)))
            before = outside_torch()
            for t in (0, len(w.fields) // 2, len(w.fields) - 1):
                sim.set_field(*w.fields[t], t); sim.relax()
            sim.set_local_field(None); sim.set_local_field(np.zeros((w.N, 2)))
            sim.sweep(w.fields[:2], step0=0)
            sim.update_fields(); sim.get_fields(0); sim.scan()
            assert sim.batch_stats()["flips"] > 0
            if attempt == 1:
                assert outside_torch() == before, "the library allocated device memory after fs_create"
                if lattice:
                    assert 0 < owned <= 3 * 4 * (8 * w.N + (1 << 20)) + 4 * w.N + (4 << 20), owned
                else:
                    assert owned == 0, owned
            sim.close(); del sim
