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
