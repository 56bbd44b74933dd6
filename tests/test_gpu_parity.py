"""GPU <-> oracle parity through the C-ABI on the five configs (scaled so the oracle
finishes in seconds) and on the edge cases.  Integer counters and the per-particle
fingerprint checksum exactly; every tally bin within 1e-9 relative."""
import numpy as np
import pytest

import mcdc_inputs as mi
from parity import compare

pytestmark = pytest.mark.gpu


def both(cfg, bank_capacity_factor=0.0, **run):
    from oracle import Oracle
    from paper_2305_07636_b200 import Problem
    o = Oracle(cfg).run(**run)
    g = Problem(cfg).run(bank_capacity_factor=bank_capacity_factor, **run)
    return g, o


CASES = {
    "config1": lambda: mi.config1(),
    "config1_3batch": lambda: mi.config1(n_hist=30_001, n_batch=3, seed=7),
    "config3_5batch": lambda: mi.config3(n_hist=10_000, n_batch=5, seed=3),       # small batches: 5 in flight
    "config3_11batch": lambda: mi.config3(n_hist=5_000, n_batch=11, seed=5),      # ... 8 in flight, 11 batches over them
    "config2": lambda: mi.config2(n_hist=100_003),
    "config3": lambda: mi.config3(n_hist=100_000),
    "config3_comb_up": lambda: mi.config3(n_hist=20_000, comb_target=33_333),
    "config3_comb_down": lambda: mi.config3(n_hist=50_000, comb_target=7_777),
    "config3_nocomb": lambda: mi.config3(n_hist=40_000, comb_target=0),
    "config4": lambda: mi.config4(n_hist=50_000, n_batch=2),
    "config4_census": lambda: mi.config4(n_hist=30_000, n_batch=1, t_end=1e-6),
    "config5_16": lambda: mi.config5(n_hist=20_000, n_batch=2, n_vox=16, n_steps=5, nusf_scale=1.0),
    "config5_64": lambda: mi.config5(n_hist=20_000, n_batch=1, nusf_scale=1.0),
    "slab_beam": lambda: mi.slab([1.0], [0.0], [0.0, 3.0], src_x=0.0, beam=True, n_hist=50_000),
    "paper_c1.1": lambda: mi.infinite_medium(1.0, 0.6, 0.2, 0.2, 2.5, 1.0, t_edges=[0.0, 20.0],
                                             t_census=[20.0], n_hist=3_000),
}


@pytest.mark.parametrize("name", list(CASES))
def test_parity(name):
    cfg = CASES[name]()
    # the c = 1.1 problem multiplies its population by e^2 inside one census step
    g, o = both(cfg, bank_capacity_factor=24.0 if name == "paper_c1.1" else 0.0)
    compare(g, o, cfg["run"]["n_batch"], o.n_steps, name)
    assert g.counters(0)["flights"] > 0


def test_tiny_and_ragged_sizes():
    for n in (1, 31, 32, 33, 255, 257):
        cfg = mi.config2(n_hist=n)
        g, o = both(cfg)
        compare(g, o, 1, o.n_steps, f"n={n}")


def test_device_tally_read_matches_host():
    from paper_2305_07636_b200 import Problem
    g = Problem(mi.config2(n_hist=5000)).run()
    for which in (0, 1, 2):
        assert np.array_equal(g.tally_device(which).cpu().numpy(), g.tally(which))


def test_bank_overflow_is_reported():
    from paper_2305_07636_b200 import Problem, McdcError
    cfg = mi.infinite_medium(1.0, 0.1, 0.1, 0.8, 2.5, 1.0, t_edges=[0.0, 30.0], t_census=[30.0], n_hist=2000)
    with pytest.raises(McdcError) as e:
        Problem(cfg).run(bank_capacity_factor=1.0)
    assert e.value.status == 5


def test_create_rejects_bad_input():
    from paper_2305_07636_b200 import Problem, McdcError
    cfg = mi.config1()
    cfg["materials"]["sigma_c"] = cfg["materials"]["sigma_c"] + 0.1
    with pytest.raises(McdcError):
        Problem(cfg)
    cfg = mi.config3()
    cfg["census"]["t_census"] = cfg["census"]["t_census"] + 1e-9
    with pytest.raises(McdcError):
        Problem(cfg)


MODES = {
    "default": {},                                             # pool kernel: one persistent launch per census step
    "pool_1pipeline": {"MCDC_PIPELINES": "1"},                 # one batch in flight at a time
    "pool_4pipelines": {"MCDC_PIPELINES": "4"},                # (the default for batches of <= 2e6; config5_16 and config4 have 2 batches)
    "pool_8pipelines": {"MCDC_PIPELINES": "8"},
    "pool_2blocks": {"MCDC_POOL_GRID": "2"},                   # few warps: long pools, children spill to the bank
    "pool_march": {"MCDC_MARCH": "1"},                         # tally marches suspended and regrouped (where the mesh is finer than the lattice)
    "pool_no_march": {"MCDC_MARCH": "0"},
    "pool_march_2blocks": {"MCDC_MARCH": "1", "MCDC_POOL_GRID": "2"},
    "pool_general": {"MCDC_LEAN": "0"},                        # the general pool kernel also where the lean variants apply (config3, config5_16)
    "events": {"MCDC_POOL": "0"},                              # per-event kernels: refill + collide + tail
    "refill_only": {"MCDC_POOL": "0", "MCDC_TAIL": "0"},       # every iteration through the refill kernel
    "plain_4flights": {"MCDC_POOL": "0", "MCDC_REFILL": "0", "MCDC_TAIL": "0"},  # block-strided multi-flight kernel
    "plain_1flight": {"MCDC_POOL": "0", "MCDC_REFILL": "0", "MCDC_MAX_FLIGHTS": "1", "MCDC_TAIL": "0"},
    "fused_bulk": {"MCDC_POOL": "0", "MCDC_FUSE_BULK": "1", "MCDC_TAIL": "0"},
    "tail_only": {"MCDC_POOL": "0", "MCDC_TAIL": "100000000"},  # whole step in the persistent work-queue kernel
}


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("name", ["config3", "config4_census", "config5_16", "config2"])
def test_parity_in_every_kernel_mode(name, mode, monkeypatch):
    """The driver picks kernels by queue length; each variant alone must reproduce the oracle."""
    for k, v in MODES[mode].items():
        monkeypatch.setenv(k, v)
    cfg = CASES[name]()
    g, o = both(cfg, bank_capacity_factor=3.0)
    compare(g, o, cfg["run"]["n_batch"], o.n_steps, f"{name}/{mode}")


@pytest.mark.parametrize("name", ["config3", "config5_16", "config5_16_tc"])
def test_lean_kernel_slow_march(name, monkeypatch):
    """Lean pool variants (tally planes = lattice planes, no pins): a flight the single-segment path cannot score (a
    particle exactly on a plane of its cell, heading out: a rounding coincidence) marches alone in march_alone().
    MCDC_LEAN=2 sends EVERY flight that way; the result must still be the oracle's."""
    monkeypatch.setenv("MCDC_LEAN", "2")
    cfg = CASES[name[:-3]]() if name.endswith("_tc") else CASES[name]()
    if name.endswith("_tc"):
        cfg["tally"]["time_crossing"] = 1
    g, o = both(cfg, bank_capacity_factor=3.0)
    assert g.kernel_path() == "pool"
    compare(g, o, cfg["run"]["n_batch"], o.n_steps, name)


@pytest.mark.parametrize("src", ["corner_isotropic", "axis_beam", "diagonal_beam", "edge_beam"])
def test_plane_ranking_degenerate_starts(src):
    """The lean pool variants rank the three plane distances of a flight without dividing and divide once
    (nearest_plane); where the ranking is not certain they take the definition's three divisions.  Sources that start
    every history in such a case: on a lattice corner (three distances of 0), along an axis (two direction cosines of
    exactly 0), along a face diagonal from a corner (two equal distances: the earlier axis wins), along an edge."""
    cfg = mi.config5(n_hist=20_000, n_batch=1, n_vox=16, n_steps=3, nusf_scale=1.0)
    s = cfg["source"]
    s["kind"] = 0
    s["lo"] = np.array([8.0, 8.0, 8.0]); s["hi"] = s["lo"].copy()
    if src == "corner_isotropic":
        s["isotropic"] = 1
    else:
        s["isotropic"] = 0
        s["dir"] = {"axis_beam": np.array([0.0, -1.0, 0.0]),
                    "diagonal_beam": np.array([np.sqrt(0.5), np.sqrt(0.5), 0.0]),
                    "edge_beam": np.array([0.0, 0.0, 1.0])}[src]
        if src == "edge_beam":
            s["lo"] = np.array([8.0, 8.0, 7.5]); s["hi"] = s["lo"].copy()
    g, o = both(cfg, bank_capacity_factor=3.0)
    compare(g, o, 1, o.n_steps, src)


def test_tail_kernel_publication_region_overflows_into_next_launch(monkeypatch):
    """Per-event path, whole step in the persistent work-queue kernel, subcritical multiplying medium
    (k = 0.9: ~5 banked children per source particle).  Lanes recycle the bank slots of particles that
    ended, so one launch can publish more children than the published region (= bank capacity) holds;
    the excess waits in a list the next launch takes.  (A smaller bank overflows for real: reported.)"""
    from paper_2305_07636_b200 import McdcError
    monkeypatch.setenv("MCDC_POOL", "0")
    monkeypatch.setenv("MCDC_TAIL", "100000000")
    N = 3_000
    cfg = mi.infinite_medium(1.0, 0.2, 0.512, 0.288, 2.5, n_hist=N)
    seen = []
    for factor in (1.5, 2.5, 3.5, 4.5, 6.0):
        try:
            g, o = both(cfg, bank_capacity_factor=factor)
        except McdcError as e:
            assert e.status == 5                       # MCDC_EOVERFLOW: the bank itself is too small
            seen.append((factor, "overflow"))
            continue
        compare(g, o, 1, o.n_steps, f"tail_only k=0.9 factor {factor}")
        c = g.counters(0)
        seen.append((factor, g.stats()["iterations"], c["secondaries"], int(factor * N) + 1024))
        assert g.kernel_path() == "events"
        if g.stats()["iterations"] >= 2:               # a second launch took the children the first could not publish
            return
    raise AssertionError(f"no bank size exercised the spill list: {seen}")


def test_pool_spill_and_relaunch(monkeypatch):
    """One block of pools (768 slots) on a strongly multiplying medium: pools fill up with fission
    parents, unborn children are handed to the bank and the kernel is relaunched over them; the
    result must still be the oracle's."""
    monkeypatch.setenv("MCDC_POOL_GRID", "1")
    cfg = mi.infinite_medium(1.0, 0.1, 0.1, 0.8, 2.5, 1.0, t_edges=[0.0, 6.0, 7.0], t_census=[6.0, 7.0],
                             n_hist=300)
    g, o = both(cfg, bank_capacity_factor=4000.0)
    compare(g, o, 1, o.n_steps, "pool spill")
    assert g.kernel_path() == "pool"
    assert g.stats()["iterations"] > o.n_steps, g.stats()      # at least one relaunch over spilled children
    assert g.counters(0)["secondaries"] > 100 * 300


def test_many_groups_upscatter_and_table_fallback():
    """More groups than any config: 24 groups (tables in shared memory, pool kernel), the same with
    the scatter rows reversed (up-scatter: no leading zeros in the CDF rows), and 80 groups (102 KB of
    tables do not fit in shared memory: the library must fall back to the per-event kernels reading
    the tables from global memory)."""
    for G, n, path, reverse in ((24, 20_000, "pool", False), (24, 20_000, "pool", True), (80, 4_000, "events", False)):
        mats, _ = mi.seeded_materials(2, fissile=(0,), G=G, rng=np.random.default_rng(5 + G))
        if reverse:
            mats["sigma_s"] = np.ascontiguousarray(mats["sigma_s"][:, :, ::-1])
        pdf = np.zeros(G); pdf[0] = 0.5; pdf[G // 2] = 0.5
        cfg = mi.infinite_multigroup(mats, 1, pdf, n_hist=n)        # material 1: scatter + capture only
        g, o = both(cfg)
        compare(g, o, 1, o.n_steps, f"G={G} reverse={reverse}")
        assert g.kernel_path() == path
        assert g.counters(0)["scatters"] > n // 2


def _with_time_crossing(cfg):
    cfg["tally"]["time_crossing"] = 1
    return cfg


TC_CASES = {
    "infinite_fine_edges": lambda: mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, 1.0, t_edges=[0.05 * k for k in range(21)],
                                                      t_census=[0.1 * k for k in range(1, 11)], n_hist=50_000, n_batch=2),
    "config2": lambda: mi.config2(n_hist=60_001),                       # general march: 100 time edges inside one census step
    "config3": lambda: mi.config3(n_hist=50_000),                       # comb: weights change at every census
    "config4_census": lambda: mi.config4(n_hist=20_000, n_batch=1, t_end=1e-6),
    "config5_16": lambda: mi.config5(n_hist=20_000, n_batch=2, n_vox=16, n_steps=5, nusf_scale=1.0),
}


@pytest.mark.parametrize("name", list(TC_CASES))
def test_time_crossing_estimator_parity(name):
    """Time-crossing block of the tally (include/mcdc.h, DESIGN.md C.13): same bins, same tolerance;
    the track-length block and every counter must not notice that it is switched on."""
    cfg = _with_time_crossing(TC_CASES[name]())
    g, o = both(cfg)
    compare(g, o, cfg["run"]["n_batch"], o.n_steps, name + " time-crossing")
    assert g.tally(2).shape[0] == 2 and g.tally(2)[1].sum() > 0.0
    plain = TC_CASES[name]()
    h = __import__("paper_2305_07636_b200").Problem(plain).run()
    assert all(h.counters(b, k) == g.counters(b, k) for b in range(cfg["run"]["n_batch"]) for k in range(o.n_steps))
    a, b = h.tally(2), g.tally(2)[0]
    assert np.all(np.abs(a - b) <= 1e-9 * np.maximum(np.abs(a), np.abs(b)))


def test_time_crossing_needs_the_pool_kernel():
    from paper_2305_07636_b200 import Problem, McdcError
    mats, _ = mi.seeded_materials(2, fissile=(0,), G=80, rng=np.random.default_rng(1))
    pdf = np.zeros(80); pdf[0] = 1.0
    cfg = _with_time_crossing(mi.infinite_multigroup(mats, 1, pdf, n_hist=100))
    with pytest.raises(McdcError):
        Problem(cfg)


def test_kernel_path_switch(monkeypatch):
    from paper_2305_07636_b200 import Problem
    cfg = mi.config2(n_hist=2000)
    assert Problem(cfg).run().kernel_path() == "pool"
    monkeypatch.setenv("MCDC_POOL", "0")
    assert Problem(cfg).run().kernel_path() == "events"


def _balance(c_list, n_source, comb):
    n_in = n_source
    for c in c_list:
        assert c["lost"] == 0
        assert n_in + c["secondaries"] == c["captures"] + c["fissions"] + c["leaks"] + c["census"]
        assert c["flights"] == c["collisions"] + c["crossings"] + c["reflections"] + c["leaks"] + c["census"]
        assert c["collisions"] == c["scatters"] + c["captures"] + c["fissions"]
        n_in = c["comb_out"] if comb and c["comb_in"] else c["census"]


def test_full_size_config5_properties(monkeypatch):
    """BASELINE config 5 at its full batch size (1e7 histories, the configuration bench.py times):
    exact particle balance per census step, comb bookkeeping, and independence of the kernel
    schedule (pool kernel vs per-event kernels): identical counters and fingerprints, tallies equal
    to 1e-9.  (The oracle needs ~14 min for this size; scaled copies are compared bin by bin above.)"""
    import torch
    from paper_2305_07636_b200 import Problem
    cfg = mi.config5(n_hist=10_000_000, n_batch=1)
    g = Problem(cfg).run()
    steps = [g.counters(0, k) for k in range(g.n_steps)]
    _balance(steps, 10_000_000, comb=True)
    assert all(c["comb_out"] == 10_000_000 for c in steps[:-1]) and steps[-1]["comb_out"] == 0
    assert all(c["comb_in"] == c["census"] for c in steps[:-1])
    assert steps[0]["source"] == 10_000_000 and sum(c["segments"] for c in steps) > 1e9
    ta = g.tally_device(2).clone()
    # per time bin: only the bins of census step k are touched during step k (tally edges = census times)
    per_t = ta.sum(dim=(1, 2, 3, 4))
    assert bool((per_t > 0).all())
    monkeypatch.setenv("MCDC_POOL", "0")
    h = Problem(cfg).run()
    assert [h.counters(0, k) for k in range(h.n_steps)] == steps
    tb = h.tally_device(2)
    assert bool(((tb == 0) == (ta == 0)).all())
    rel = ((ta - tb).abs() / torch.clamp(torch.maximum(ta.abs(), tb.abs()), min=1e-300)).max().item()
    assert rel <= 1e-9, rel
    del ta, tb, g, h
    torch.cuda.empty_cache()


@pytest.mark.parametrize("pool", [1, 0])
def test_full_size_config5_against_the_oracle(pool, monkeypatch):
    """BASELINE config 5 at the batch size bench.py times (1e7 histories, seed 0, 20 census steps with
    comb), in the launch configuration bench.py uses, against what the ORACLE computed for the same
    batch (tests/golden/config5_1e7_seed0.npz, written by tests/golden/make_config5_1e7.py, which calls
    only oracle/): every counter row and fingerprint as integers, 1e5 seeded-random bins within 1e-9,
    2e4 zero bins exactly zero, the number of non-zero bins of every (time, group) plane, and the
    exactly rounded plane sums within 1e-9.  Both kernel paths."""
    import math
    import os
    import torch
    from paper_2305_07636_b200 import Problem
    from paper_2305_07636_b200.binding import COUNTER_NAMES
    gold = np.load(os.path.join(os.path.dirname(__file__), "golden", "config5_1e7_seed0.npz"))
    assert int(gold["n_hist"]) == 10_000_000
    monkeypatch.setenv("MCDC_POOL", str(pool))
    g = Problem(mi.config5(n_hist=10_000_000, n_batch=1, seed=0)).run()
    assert g.kernel_path() == ("pool" if pool else "events")
    got = np.array([[g.counters(0, k)[n] for n in COUNTER_NAMES] for k in range(g.n_steps)], dtype=np.uint64)
    bad = np.argwhere(got != gold["counters"])
    assert bad.size == 0, [(int(k), COUNTER_NAMES[int(i)], int(got[k, i]), int(gold["counters"][k, i])) for k, i in bad[:8]]
    t = g.tally_device(2)
    flat = t.reshape(-1)
    val = flat[torch.as_tensor(gold["idx"], device="cuda")].cpu().numpy()
    ref = gold["val"]
    assert np.all(val[ref == 0.0] == 0.0)
    err = np.abs(val - ref) / np.maximum(np.maximum(np.abs(val), np.abs(ref)), 1e-300)
    assert err[ref != 0.0].max() <= 1e-9, err.max()
    assert np.count_nonzero(ref) > 50_000
    assert bool((flat[torch.as_tensor(gold["zero_idx"], device="cuda")] == 0.0).all())
    nz = (t != 0).sum(dim=(2, 3, 4)).cpu().numpy()
    assert np.array_equal(nz, gold["nonzero"])
    planes = t.reshape(t.shape[0], t.shape[1], -1).cpu().numpy()
    sums = np.array([[math.fsum(planes[a, b]) for b in range(planes.shape[1])] for a in range(planes.shape[0])])
    assert np.all(np.abs(sums - gold["plane_sums"]) <= 1e-9 * np.abs(gold["plane_sums"]))
    del t, flat, g
    torch.cuda.empty_cache()


@pytest.mark.parametrize("k", [2, 3, 4])
def test_full_size_parity_configs_2_3_4(k):
    """BASELINE configs 2, 3 and 4 at their full batch size (1e6 histories; one batch), on the kernel
    path bench.py times: the oracle finishes these in seconds, so the comparison is bin by bin."""
    cfg = mi.config(k, n_hist=1_000_000, n_batch=1)
    g, o = both(cfg)
    compare(g, o, 1, o.n_steps, f"config{k} full size")
    assert g.kernel_path() == "pool" and g.counters(0)["source"] == 1_000_000


def test_config4_one_batch_of_1e7_against_the_oracle():
    """BASELINE config 4 names 1e7 histories; bench.py also times them as batches of 1e7 (two in flight,
    `--config 4 --n-hist 10000000`): one such batch against the oracle (13 s on one core), bin by bin."""
    cfg = mi.config4(n_hist=10_000_000, n_batch=1)
    g, o = both(cfg)
    compare(g, o, 1, o.n_steps, "config4 1e7")
    assert g.kernel_path() == "pool" and g.counters(0)["source"] == 10_000_000


def test_config5_full_geometry_200k():
    """Config 5 with its full geometry, tally, census schedule and calibrated fission scale at 2e5
    histories (the oracle needs ~15 s; at the full 1e7 it needs ~14 min, see the property test)."""
    cfg = mi.config5(n_hist=200_000, n_batch=1)
    g, o = both(cfg)
    compare(g, o, 1, o.n_steps, "config5 200k")
    assert g.kernel_path() == "pool"


def test_full_size_config4_properties():
    """BASELINE config 4 at full batch size (1e6 histories per batch, 2 of the 10 batches)."""
    from paper_2305_07636_b200 import Problem
    cfg = mi.config4(n_hist=1_000_000, n_batch=2)
    g = Problem(cfg).run()
    for b in range(2):
        c = g.counters(b)
        _balance([c], 1_000_000, comb=False)
        assert c["leaks"] == 0 and c["reflections"] > 0
    T = g.tally(0).sum(axis=(0, 1, 2))
    cells = T.reshape(17, 3, 17, 3).transpose(0, 2, 1, 3).sum(axis=(2, 3))
    assert cells.std() / cells.mean() < 0.02


# ---------------------------------------------------------------------------------------------
# k-eigenvalue mode (DESIGN.md §3 C.14): every generation's counters and the
# fingerprint exactly, the k of every cycle bit for bit (it is a function of integer counts and
# IEEE multiplies/divides), the active-cycle tally within 1e-9
EIG_CASES = {
    "eig_1g_infinite": lambda: mi.eigenvalue(mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, n_hist=20_000), 3, 5),
    "eig_1g_k0_half": lambda: mi.eigenvalue(mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, n_hist=5_000), 2, 3, k0=0.5),
    "eig_slab_leaking": lambda: mi.eigenvalue(mi.fissile_slab(width=6.0, n_hist=20_000, n_batch=2), 4, 6),
    "eig_pin_cell": lambda: mi.pin_cell_eigenvalue(n_hist=10_000, n_inactive=3, n_active=4, mesh=(5, 5, 10)),
    "eig_pin_cell_9batch": lambda: mi.pin_cell_eigenvalue(n_hist=4_000, n_inactive=2, n_active=3, mesh=(5, 5, 10), n_batch=9),   # eight in flight
    "eig_one_cycle": lambda: mi.eigenvalue(mi.fissile_slab(width=4.0, n_hist=3_333), 0, 1),
    "eig_delayed_7g": lambda: mi.eigenvalue(mi.seeded_delayed(mi.infinite_multigroup(mi.seeded_materials(2, fissile=(0,), nusf_scale=7.0)[0], 0,
                                                                                   mi.seeded_materials(2, fissile=(0,))[0]["chi"][0], n_hist=10_000),
                                                              J=3, beta=0.4), 2, 4),
    "eig_tiny": lambda: mi.eigenvalue(mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, n_hist=33), 1, 4),
}


@pytest.mark.parametrize("name", list(EIG_CASES))
def test_eigenvalue_parity(name):
    cfg = EIG_CASES[name]()
    # k0 = 0.5 makes the first generation bank 2.5 children per particle
    g, o = both(cfg, bank_capacity_factor=4.0 if name == "eig_1g_k0_half" else 0.0)
    assert g.n_steps == o.n_steps == cfg["eigenvalue"]["n_inactive"] + cfg["eigenvalue"]["n_active"]
    compare(g, o, cfg["run"]["n_batch"], o.n_steps, name)
    for b in range(cfg["run"]["n_batch"]):
        assert np.array_equal(g.k_cycle(b), o.k_cycle(b)), name
    c = g.counters(0, 0)
    assert c["segments"] == 0 if cfg["eigenvalue"]["n_inactive"] > 0 else c["segments"] > 0
    assert g.kernel_path() == "pool"


def test_eigenvalue_rejects_time_dependent_and_reports_die_out():
    from paper_2305_07636_b200 import Problem, McdcError
    cfg = mi.config3(n_hist=1000)
    cfg["eigenvalue"] = dict(n_inactive=1, n_active=1, k0=1.0)
    with pytest.raises(McdcError) as e:
        Problem(cfg)
    assert e.value.status == 1
    for bad in (dict(n_inactive=-1, n_active=1, k0=1.0), dict(n_inactive=0, n_active=0, k0=1.0),
                dict(n_inactive=0, n_active=1, k0=0.0)):
        cfg = mi.config1(n_hist=100)
        cfg["eigenvalue"] = bad
        with pytest.raises(McdcError):
            Problem(cfg)
    # no fissile material: the first generation has no children
    cfg = mi.eigenvalue(mi.config1(n_hist=500), 1, 2)
    with pytest.raises(McdcError) as e:
        Problem(cfg).run()
    assert e.value.status == 4
    # a first generation that more than fills the bank (k0 = 0.5: 2.5 children per particle)
    with pytest.raises(McdcError) as e:
        Problem(EIG_CASES["eig_1g_k0_half"]()).run()
    assert e.value.status == 5
    # nu / k above 7 children
    cfg = mi.eigenvalue(mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, n_hist=500), 1, 2, k0=0.25)
    with pytest.raises(McdcError) as e:
        Problem(cfg).run()
    assert e.value.status == 1


# ---------------------------------------------------------------------------------------------
# implicit capture, weight roulette, weighted comb (DESIGN.md §3 C.15)
def _ic_td_tc():
    cfg = mi.infinite_medium(1.0, 0.5, 0.3, 0.2, 2.5, 1.0, t_edges=[0.0, 1.0, 2.0, 3.0], t_census=[1.0, 2.0, 3.0],
                             comb_target=25_000, n_hist=20_000, n_batch=2)
    cfg["tally"]["time_crossing"] = 1
    return mi.implicit_capture(cfg, 0.2, 0.6)


IC_CASES = {
    "ic_config1_roulette": lambda: mi.implicit_capture(mi.config1(n_hist=50_000, n_batch=2), 0.5, 0.5),
    "ic_config2": lambda: mi.implicit_capture(mi.config2(n_hist=100_003), 0.1, 0.3),
    "ic_config3_wcomb": lambda: mi.implicit_capture(mi.config3(n_hist=50_000), 0.0, 1.0),
    "ic_config3_wcomb_roulette": lambda: mi.implicit_capture(mi.config3(n_hist=30_000, comb_target=41_111), 0.4, 0.8),
    "ic_config3_wcomb_down": lambda: mi.implicit_capture(mi.config3(n_hist=30_000, comb_target=7_777), 0.3, 0.3),
    "ic_config4": lambda: mi.implicit_capture(mi.config4(n_hist=30_000, n_batch=2), 0.25, 0.5),
    "ic_config5_16": lambda: mi.implicit_capture(mi.config5(n_hist=20_000, n_batch=2, n_vox=16, n_steps=5, nusf_scale=1.0), 0.25, 0.75),
    "ic_time_crossing_wcomb": _ic_td_tc,
    "ic_tiny": lambda: mi.implicit_capture(mi.config3(n_hist=33, comb_target=40), 0.3, 0.6),
}


@pytest.mark.parametrize("name", list(IC_CASES))
def test_implicit_capture_parity(name):
    cfg = IC_CASES[name]()
    g, o = both(cfg)
    compare(g, o, cfg["run"]["n_batch"], o.n_steps, name)
    assert g.kernel_path() == "pool"
    if cfg["census"]["comb_target"]:
        assert g.counters(0, 0)["comb_out"] == cfg["census"]["comb_target"]


def test_implicit_capture_rejects_bad_arguments():
    from paper_2305_07636_b200 import Problem, McdcError
    for bad in ((-1.0, 1.0), (0.5, 0.25), (0.1, 1e9)):
        with pytest.raises(McdcError) as e:
            Problem(mi.implicit_capture(mi.config1(n_hist=10), *bad))
        assert e.value.status == 1
    with pytest.raises(McdcError):
        Problem(mi.eigenvalue(mi.implicit_capture(mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, n_hist=10)), 1, 1))


def test_full_size_eigenvalue_paper_run():
    """The paper's k-eigenvalue run shape (50 inactive + 100 active cycles of 1e5
    particles, 20 x 20 x 100 x 7 tally) on the pin-cell stand-in, the configuration
    `bench.py --eigenvalue 50,100` times: every cycle's counters, fingerprint and k bit for bit, the
    280 000-bin active-cycle tally within 1e-9 (the oracle needs ~20 s)."""
    cfg = mi.pin_cell_eigenvalue(n_hist=100_000, n_inactive=50, n_active=100)
    g, o = both(cfg)
    compare(g, o, 1, 150, "pin-cell eigenvalue 50+100 x 1e5")
    assert np.array_equal(g.k_cycle(), o.k_cycle())
    k = g.k_cycle()[50:]
    assert abs(k.mean() - 1.0) < 0.05 and k.std() < 0.02


def test_full_size_implicit_capture_config3():
    """Config 3 at its full size (1e6 histories, 20 census steps, comb to 1e6) with implicit capture,
    the roulette and the weighted comb: bin by bin and counter by counter against the oracle."""
    cfg = mi.implicit_capture(mi.config3(n_hist=1_000_000), 0.25, 0.5)
    g, o = both(cfg)
    compare(g, o, 1, o.n_steps, "config3 full size, implicit capture")
    assert all(g.counters(0, k)["comb_out"] == 1_000_000 for k in range(19))


# ---------------------------------------------------------------------------------------------
# delayed neutrons (DESIGN.md §3 C.16)
def _dn_kinetics(comb=0, tc=0, n_hist=20_000, n_batch=2):
    tk = np.linspace(0.0, 4.0, 9)
    cfg = mi.infinite_medium(1.0, 0.4, 0.35, 0.25, 2.4, 1.0, t_edges=tk, t_census=tk[1:], comb_target=comb,
                             n_hist=n_hist, n_batch=n_batch)
    cfg["tally"]["time_crossing"] = tc
    return mi.delayed(cfg, [[[0.6, 0.3]]], [[0.8, 3.0]])


DN_CASES = {
    "dn_point_kinetics": lambda: _dn_kinetics(),
    "dn_comb": lambda: _dn_kinetics(comb=23_456),
    "dn_time_crossing_comb": lambda: _dn_kinetics(comb=20_000, tc=1),
    "dn_time_independent": lambda: mi.delayed(mi.infinite_medium(1.0, 0.4, 0.4, 0.2, 2.0, n_hist=30_000, n_batch=2),
                                              [[[0.5, 0.2]]], [[0.1, 2.0]]),
    "dn_config4_census": lambda: mi.seeded_delayed(mi.config4(n_hist=30_000, n_batch=1, t_end=1e-6), beta=0.3, time_scale=1e-6),
    "dn_config4": lambda: mi.seeded_delayed(mi.config4(n_hist=20_000, n_batch=2), beta=0.3, time_scale=1e-5),
    "dn_config5_16": lambda: mi.seeded_delayed(mi.config5(n_hist=20_000, n_batch=2, n_vox=16, n_steps=5, nusf_scale=1.0),
                                               beta=0.2, time_scale=1e-6),
    "dn_tiny": lambda: _dn_kinetics(comb=40, n_hist=33, n_batch=1),
}


@pytest.mark.parametrize("name", list(DN_CASES))
def test_delayed_neutron_parity(name):
    cfg = DN_CASES[name]()
    g, o = both(cfg)
    compare(g, o, cfg["run"]["n_batch"], o.n_steps, name)
    assert g.kernel_path() == "pool"
    c = g.counters(0)
    if len(cfg["census"]["t_census"]) > 1:
        assert c["flights"] > c["collisions"] + c["crossings"] + c["reflections"] + c["leaks"]   # census events incl. waiting


def test_delayed_rejects_bad_arguments():
    from paper_2305_07636_b200 import Problem, McdcError
    base = mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, n_hist=10)
    for nud, lam, chd in (([[[2.0, 1.0]]], [[0.5, 2.0]], None), ([[[0.4, 0.3]]], [[0.5, 0.0]], None),
                          ([[[0.4, 0.3]]], [[0.5, 2.0]], [[[0.9], [1.0]]])):
        with pytest.raises(McdcError) as e:
            Problem(mi.delayed(base, nud, lam, chd))
        assert e.value.status == 1


# ---------------------------------------------------------------------------------------------
# source with a time extent (DESIGN.md §3 C.17) and the dog-leg duct stand-in of the
# paper's time-dependent Kobayashi run (source window + implicit capture + mesh tally)
def _sw_infinite():
    tk = np.linspace(0.0, 4.0, 9)
    cfg = mi.infinite_medium(1.0, 0.5, 0.5, 0.0, 0.0, 1.0, t_edges=tk, t_census=tk[1:], n_hist=30_000, n_batch=2)
    cfg["source"]["t_end"] = 2.0
    return cfg


def _sw_dn_ic():
    cfg = _dn_kinetics(comb=20_000)
    cfg["source"] = dict(cfg["source"]); cfg["source"]["t_end"] = 1.3
    return mi.implicit_capture(cfg, 0.2, 0.5)


SW_CASES = {
    "sw_infinite": _sw_infinite,
    "sw_dogleg_analog": lambda: mi.dogleg_duct(n_hist=50_000, n_batch=2),
    "sw_dogleg_ic": lambda: mi.implicit_capture(mi.dogleg_duct(n_hist=20_000), 0.0, 1.0),
    "sw_dogleg_ic_roulette": lambda: mi.implicit_capture(mi.dogleg_duct(n_hist=30_000, n_census=10), 0.1, 0.5),
    "sw_delayed_ic_wcomb": _sw_dn_ic,
}


@pytest.mark.parametrize("name", list(SW_CASES))
def test_source_window_parity(name):
    cfg = SW_CASES[name]()
    g, o = both(cfg)
    compare(g, o, cfg["run"]["n_batch"], o.n_steps, name)
    assert g.kernel_path() == "pool"
    c = g.counters(0)
    assert c["flights"] > c["collisions"] + c["crossings"] + c["reflections"] + c["leaks"]


def test_c_abi_from_plain_c(tmp_path):
    """The boundary without Python or torch: tests/helpers/abi_c_smoke.c is compiled with gcc against
    include/mcdc.h, linked with the in-tree library and the CUDA runtime, and runs config 1 (flux =
    1/Sigma_a = 2, every history ends in a capture)."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    from paper_2305_07636_b200.build import build
    lib = build()
    exe = tmp_path / "abi_c_smoke"
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    subprocess.run(["gcc", "-std=c11", "-O1", "-I", os.path.join(root, "include"), "-I", os.path.join(cuda, "include"),
                    os.path.join(root, "tests", "helpers", "abi_c_smoke.c"), "-o", str(exe), lib,
                    "-L", os.path.join(cuda, "lib64"), "-lcudart", "-lm",
                    "-Wl,-rpath," + os.path.dirname(lib), "-Wl,-rpath," + os.path.join(cuda, "lib64")], check=True)
    r = subprocess.run([str(exe)], capture_output=True, text=True)
    assert r.returncode == 0 and r.stdout.strip().endswith("OK"), r.stdout + r.stderr


# ---------------------------------------------------------------------------------------------
# every combination of the options (time-crossing block, implicit capture, delayed neutrons, source
# window, comb) on a 1-group kinetics problem and on the 7-group pin lattice: each combination runs its
# own instantiation of the pool kernel / census close
def _combo(base, tc, ic, dn, window, comb):
    if base == "kinetics":
        tk = np.linspace(0.0, 3.0, 7)
        cfg = mi.infinite_medium(1.0, 0.4, 0.35, 0.25, 2.4, 1.0, t_edges=tk, t_census=tk[1:],
                                 comb_target=9_000 if comb else 0, n_hist=8_000, n_batch=2)
        if dn:
            cfg = mi.delayed(cfg, [[[0.6, 0.3]]], [[0.8, 3.0]])
        t_win = 1.2
    else:
        cfg = mi.config4(n_hist=6_000, n_batch=2, t_end=1e-6)
        tt = cfg["tally"]["tts"]
        cfg["census"] = dict(t_census=tt[[3, 7, 10]].copy(), comb_target=7_000 if comb else 0)
        if dn:
            cfg = mi.seeded_delayed(cfg, beta=0.3, time_scale=1e-6)
        t_win = 4e-7
    cfg["tally"] = dict(cfg["tally"]); cfg["tally"]["time_crossing"] = int(tc)
    if window:
        cfg["source"] = dict(cfg["source"]); cfg["source"]["t_end"] = t_win
    if ic:
        cfg = mi.implicit_capture(cfg, 0.2, 0.5)
    return cfg


import itertools  # noqa: E402


@pytest.mark.parametrize("base", ["kinetics", "pins"])
@pytest.mark.parametrize("tc,ic,dn,window,comb", [c for c in itertools.product((0, 1), repeat=5) if sum(c) >= 2])
def test_option_combinations(base, tc, ic, dn, window, comb):
    cfg = _combo(base, tc, ic, dn, window, comb)
    g, o = both(cfg, bank_capacity_factor=3.0)
    compare(g, o, 2, o.n_steps, f"{base} tc={tc} ic={ic} dn={dn} window={window} comb={comb}")


@pytest.mark.parametrize("tc,ic,dn,window,comb", [c for c in itertools.product((0, 1), repeat=5) if sum(c) >= 2])
def test_option_combinations_with_regrouped_marches(tc, ic, dn, window, comb, monkeypatch):
    """The same option combinations on the pin lattice (tally mesh finer than the lattice) in the kernel
    variants that suspend and regroup tally marches, which a run otherwise takes only after a batch has
    counted many segments per flight."""
    monkeypatch.setenv("MCDC_MARCH", "1")
    cfg = _combo("pins", tc, ic, dn, window, comb)
    g, o = both(cfg, bank_capacity_factor=3.0)
    compare(g, o, 2, o.n_steps, f"pins/march tc={tc} ic={ic} dn={dn} window={window} comb={comb}")


def test_march_variant_is_taken_after_a_batch_with_long_marches():
    """Batches after the first follow the segments per flight the finished ones counted: config 2 (12
    segments per flight) switches to the regrouping variants, and every batch still equals the oracle."""
    cfg = mi.config2(n_hist=60_000, n_batch=3)
    g, o = both(cfg)
    compare(g, o, 3, o.n_steps, "config2 3 batches, adaptive march")
    c = g.counters(0)
    assert c["segments"] > 6 * c["flights"]
    # eigenvalue pin cell with the regrouping variants forced
    import os
    os.environ["MCDC_MARCH"] = "1"
    try:
        cfg = mi.pin_cell_eigenvalue(n_hist=5_000, n_inactive=2, n_active=3, mesh=(5, 5, 10))
        g, o = both(cfg)
        compare(g, o, 1, o.n_steps, "eig pin cell, march")
        assert np.array_equal(g.k_cycle(0), o.k_cycle(0))
    finally:
        del os.environ["MCDC_MARCH"]


# ---------------------------------------------------------------------------------------------
# C.1: a particle that reaches 2^24 - 1 flights under one id ends as lost (its streams would repeat)
def test_flight_counter_limit_is_reported_as_lost():
    from oracle import Oracle
    from paper_2305_07636_b200 import Problem, McdcError
    cfg = mi.infinite_medium(1.0, 1.0, 0.0, n_hist=2)           # a pure scatterer: histories never end
    o = Oracle(cfg)
    with pytest.raises(RuntimeError):
        o.run()
    g = Problem(cfg)
    with pytest.raises(McdcError) as e:
        g.run()
    assert e.value.status == 6
    cg, co = g.counters(0), o.counters(0)
    assert cg == co and cg["lost"] == 2 and cg["flights"] == 2 * (1 << 24) and cg["scatters"] == 2 * ((1 << 24) - 1)
    assert g.tally(2).item() == pytest.approx(o.tally(2).item(), rel=1e-9)


# ---------------------------------------------------------------------------------------------
# Replicas (include/mcdc.h mcdc_replica_layout / mcdc_replica_commit): two "ranks" on one
# GPU, one after the other; the sum all-reduce is stood in for by adding rank 1's sums and counters into
# rank 0's workspace views (what NCCL does in place); the committed result equals one run of all batches.
def test_replica_combine_equals_one_run_of_all_batches():
    import torch
    from paper_2305_07636_b200 import Problem, replicas
    cfg = mi.config2(n_hist=20_000, n_batch=2)
    whole = Problem(cfg).run(seed=10, n_batch=4)
    r0 = Problem(cfg).run(seed=10, n_batch=2)
    r1 = Problem(cfg).run(seed=12, n_batch=2)
    s0, c0 = r0.replica_views()
    s1, c1 = r1.replica_views()
    s0 += s1; c0 += c1
    torch.cuda.synchronize()
    r0.replica_commit(2)
    np.testing.assert_allclose(r0.tally(0), whole.tally(0), rtol=1e-12, atol=0)
    se, se_ref = r0.tally(1), whole.tally(1)
    mean = whole.tally(0)
    assert np.all(np.abs(se * se - se_ref * se_ref) <= 4e-9 * mean * mean + 1e-300)
    for b in range(2):
        a, b0, b1 = r0.counters(b), whole.counters(b), whole.counters(b + 2)
        assert all(a[n] == (b0[n] + b1[n]) % (1 << 64) for n in a)
    # world size 1: combine is the commit alone and changes nothing
    w2 = replicas.combine(Problem(cfg).run(seed=10, n_batch=4))
    # (equal up to the order in which the pipelines folded their batches into the sums)
    np.testing.assert_allclose(w2.tally(0), whole.tally(0), rtol=1e-12, atol=0)
    np.testing.assert_allclose(w2.tally(1), whole.tally(1), rtol=1e-6, atol=1e-300)


# ---------------------------------------------------------------------------------------------
# Quadric-surface CSG (C.18) and moving surfaces (C.19): counters, fingerprints and tallies as everywhere
def _csg_shells(n_hist=30_000, census=False, comb=0, motion=False, tilt=True, **kw):
    """A sphere, a shell around it, a tilted cylinder through both and a cutting plane in a reflective /
    vacuum box of 7-group materials: nested and overlapping regions, eleven of them."""
    mats, _ = mi.seeded_materials(3, fissile=(0,), nusf_scale=1.5)
    S = [mi.quadric_sphere((0.2, -0.1, 0.3), 1.1),                      # 1
         mi.quadric_sphere((0.2, -0.1, 0.3), 2.0),                      # 2
         mi.quadric_cylinder((0.0, 0.0, 0.0), (1.0, 2.0, 0.5) if tilt else (0, 0, 1), 0.7),   # 3
         mi.quadric_plane((0.3, -0.5, 1.0), 0.4),                       # 4
         mi.quadric_general(np.diag([1.0, 0.5, -1.0]), [0, 0, 0], -6.0)]   # 5: hyperboloid of one sheet
    R = [([-1, -3], 0), ([-1, 3, -4], 1), ([-1, 3, 4], 2),
         ([1, -2, -3], 1), ([1, -2, 3, -4], 0), ([1, -2, 3, 4], 2),
         ([2, -3, -5], 2), ([2, -3, 5], 1), ([2, 3, -5, -4], 1), ([2, 3, -5, 4], 0), ([2, 3, 5], 2)]
    tt = np.array([0.0, 2e-9, 5e-9, 1e-8, 3e-8]) if census else np.array([0.0, mi.INF])
    tally = dict(txs=np.linspace(-4, 4, 9), tys=np.linspace(-4, 4, 5), tzs=np.linspace(-4, 4, 7), tts=tt)
    pdf = np.zeros(7); pdf[0] = 0.6; pdf[2] = 0.4
    src = mi.ball_source((0.2, -0.1, 0.3), 1.5, G=7); src["group_pdf"] = pdf
    mv = None
    if motion:
        tau = [1e-9, 4e-9, 2e-8]
        disp = np.zeros((5, 3, 3))
        disp[0, 1] = (0.3, 0.0, -0.2); disp[0, 2] = (0.3, 0.4, -0.2)       # the inner sphere moves, then turns
        disp[3, :, 2] = (0.0, 0.5, -0.3)                                   # the plane goes up and comes back down
        mv = (tau, disp)
    return mi.csg_problem(mats, S, R, box=((-4, 4),) * 3, bc=(1, 0, 1, 1, 0, 1), source=src, tally=tally,
                          t_census=tt[1:] if census else (), comb_target=comb, n_hist=n_hist, motion=mv, name="csg_shells", **kw)


def _csg_tc():
    c = _csg_shells(census=True, comb=25_000, n_hist=20_000); c["tally"]["time_crossing"] = 1
    return c


CSG_CASES = {
    "csg_shells": lambda: _csg_shells(),
    "csg_census_comb": lambda: _csg_shells(census=True, comb=30_000),
    "csg_moving": lambda: _csg_shells(census=True, comb=0, motion=True, n_hist=20_000, n_batch=2),
    "csg_moving_comb_tc": lambda: (lambda c: (c["tally"].__setitem__("time_crossing", 1), c)[1])(_csg_shells(census=True, comb=20_000, motion=True, n_hist=20_000)),
    "csg_time_crossing": _csg_tc,
    "csg_implicit_capture": lambda: mi.implicit_capture(_csg_shells(census=True, comb=20_000, n_hist=20_000), 0.2, 0.5),
    "csg_delayed": lambda: mi.seeded_delayed(_csg_shells(census=True, comb=20_000, n_hist=20_000), beta=0.3, time_scale=1e-9),
    "csg_slab_planes": lambda: (lambda ref: mi.csg_problem(ref["materials"], [mi.quadric_plane((1, 0, 0), x) for x in (5.0, 10.0, 15.0)],
                                                          [([-1], 0), ([1, -2], 1), ([2, -3], 2), ([3], 3)],
                                                          box=((0.0, 20.0), (-mi.INF, mi.INF), (-mi.INF, mi.INF)), source=ref["source"],
                                                          tally=ref["tally"], t_census=ref["census"]["t_census"], n_hist=50_000))(mi.config2(n_hist=10)),
    "csg_moving_interface": lambda: mi.csg_problem(mi._materials_1g([0.7, 1e-9], [0.3, 0.0], [0.4, 1e-9], [0, 0], [0, 0], speed=2.0),
                                                   [mi.quadric_plane((1, 0, 0), 3.0)], [([-1], 1), ([1], 0)],
                                                   box=((-20.0, 20.0), (-mi.INF, mi.INF), (-mi.INF, mi.INF)),
                                                   tally=dict(txs=np.linspace(-20, 20, 41), tys=np.array([-mi.INF, mi.INF]),
                                                              tzs=np.array([-mi.INF, mi.INF]), tts=np.linspace(0, 6, 13)),
                                                   t_census=[2.0, 4.0, 6.0], n_hist=20_000,
                                                   motion=([0.0, 1.0, 11.0], [[[0, 0, 0], [1.5, 0, 0], [6.5, 0, 0]]])),
    "csg_tiny": lambda: _csg_shells(n_hist=33),
}


@pytest.mark.parametrize("name", list(CSG_CASES))
def test_quadric_csg_parity(name):
    cfg = CSG_CASES[name]()
    g, o = both(cfg, bank_capacity_factor=4.0)
    compare(g, o, cfg["run"]["n_batch"], o.n_steps, name)
    c = g.counters(0)
    assert g.kernel_path() == "pool" and c["crossings"] > 0 and c["lost"] == 0
    if "moving" in name:
        assert cfg["motion"]["tau"].size >= 2


def test_quadric_csg_hole_and_bad_arguments():
    from oracle import Oracle
    from paper_2305_07636_b200 import Problem, McdcError
    hole = mi.csg_problem(mi._materials_1g([1e-9], [0.0], [1e-9], [0], [0]), [mi.quadric_sphere((0, 0, 0), 1.0)],
                          [([-1], 0)], box=((-5, 5),) * 3, n_hist=1000)
    o = Oracle(hole)
    with pytest.raises(RuntimeError):
        o.run()
    g = Problem(hole)
    with pytest.raises(McdcError) as e:
        g.run()
    assert e.value.status == 6 and g.counters(0) == o.counters(0) and g.counters(0)["lost"] == 1000
    lat = mi.config2(n_hist=10); lat["csg"] = hole["csg"]
    with pytest.raises(McdcError):
        Problem(lat)
    bad = dict(hole); bad["csg"] = dict(hole["csg"]); bad["csg"]["region_mat"] = np.array([2], np.int32)
    with pytest.raises(McdcError):
        Problem(bad)
    ball = mi.config1(n_hist=10); ball["source"] = mi.ball_source((0, 0, 0), 1.0)
    with pytest.raises(McdcError):
        Problem(ball).run()
    eig = mi.eigenvalue(dict(hole), 1, 2)
    with pytest.raises(McdcError):
        Problem(eig)
