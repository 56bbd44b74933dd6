"""Closed-form, invariant and special-case pins of the oracle's transport loop
(P3-P11, P15, P16; BASELINE.json north_star: S/Sigma_a, exp(-Sigma_t L),
exp((nu Sigma_f - Sigma_a) v t), particle balance, each within 4 sigma)."""
import math

import numpy as np
import pytest

import mcdc_inputs as mi
from oracle import Oracle


def balance_ok(o, batch=0):
    """P7: N_in + secondaries == captures + fissions + leaks + census, per census step."""
    n_in = o.counters(batch, 0)["source"]
    for k in range(o.n_steps):
        c = o.counters(batch, k)
        assert c["lost"] == 0
        assert n_in + c["secondaries"] == c["captures"] + c["fissions"] + c["leaks"] + c["census"]
        assert c["flights"] == c["collisions"] + c["crossings"] + c["reflections"] + c["leaks"] + c["census"]
        assert c["collisions"] == c["scatters"] + c["captures"] + c["fissions"]
        if k + 1 < o.n_steps:
            n_in = c["comb_out"] if c["comb_out"] or c["comb_in"] else c["census"]
            if c["comb_in"]:
                assert c["comb_in"] == c["census"]


def test_config1_flux_is_S_over_sigma_a():
    """P3 (BASELINE.json:7): flux per source particle = 1/Sigma_a = 2; track length ~ Exp, var 4."""
    N = 100_000
    o = Oracle(mi.config1(n_hist=N)).run()
    c = o.counters()
    flux = o.tally(0).item()
    assert abs(flux - 2.0) < 4 * 2.0 / math.sqrt(N)
    assert c["captures"] == N and c["leaks"] == 0 and c["census"] == 0 and c["fissions"] == 0
    assert abs(c["collisions"] / N - 2.0) < 4 * math.sqrt(2.0 / N)
    assert c["segments"] == c["flights"] == c["collisions"]
    balance_ok(o)


def test_absorbing_slab_transmission():
    """P4: beam on a purely absorbing slab, L = 3: leaks/N = exp(-3); uncollided flux integral."""
    N = 200_000
    cfg = mi.slab([1.0], [0.0], [0.0, 3.0], src_x=0.0, beam=True, n_hist=N)
    o = Oracle(cfg).run()
    c = o.counters()
    p = math.exp(-3.0)
    assert abs(c["leaks"] / N - p) < 4 * math.sqrt(p * (1 - p) / N)
    assert c["scatters"] == 0 and c["captures"] + c["leaks"] == N
    # track length per particle = min(Exp(1), 3): mean 1 - e^-3, var = 1 - 2*3*e^-3 - e^-6
    mean = 1 - p
    var = 1 - 6 * p - p * p
    assert abs(o.tally(0).item() - mean) < 4 * math.sqrt(var / N)
    balance_ok(o)


@pytest.mark.parametrize("comb", [0, 1])
def test_config3_growth(comb):
    """P5 (BASELINE.json:9): alpha = v (nu Sigma_f - Sigma_a) = 0.15; interval flux
    (e^{a t_k} - e^{a t_{k-1}})/a per source particle; pre-comb population ratio e^{0.015}."""
    N = 200_000
    o = Oracle(mi.config3(n_hist=N, comb_target=N if comb else 0)).run()
    a = 0.15
    tk = np.array([0.1 * k for k in range(21)])
    expect = (np.exp(a * tk[1:]) - np.exp(a * tk[:-1])) / a
    got = o.tally(0).ravel()
    # std of the population at t is <~ sqrt(c t / N) with c = O(1); 4 sigma bound, generous constant
    tol = 4 * expect * np.sqrt((0.5 + 2.0 * tk[1:]) / N)
    assert np.all(np.abs(got - expect) < tol), (got - expect) / tol
    if comb:
        ratios = np.array([o.counters(0, k)["comb_in"] / N for k in range(19)])
        assert np.all(np.abs(ratios - math.exp(0.015)) < 4 * math.sqrt(0.04 / N))
        assert all(o.counters(0, k)["comb_out"] == N for k in range(19))
    else:
        pop = o.counters(0, 19)["census"] / N
        assert abs(pop - math.exp(0.3)) < 4 * math.exp(0.3) * math.sqrt(2.5 / N)
    balance_ok(o)


def test_paper_worked_value_population_7_39():
    """P6 (fixture tests/golden/paper_values.txt): c = 1.1 -> population x e^2 = 7.39
    after 20 mean free times."""
    import os
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()[:2]; vals[k] = float(v)
    N = 40_000
    # Sigma_t = 1, v = 1: Sigma_s 0.6 + nu Sigma_f = 2.5 * 0.2 = 0.5 -> c = 1.1; capture 0.2
    cfg = mi.infinite_medium(1.0, 0.6, 0.2, 0.2, 2.5, 1.0, t_edges=[0.0, 20.0], t_census=[20.0], n_hist=N)
    o = Oracle(cfg).run()
    pop = o.counters()["census"] / N
    assert abs(vals["azurv1_growth_20mft"] - math.exp(2.0)) < 0.005     # the paper's "about 7.39" is e^2
    assert abs(pop - math.exp(2.0)) < 4 * math.exp(2.0) * math.sqrt(12.0 / N)
    assert abs(pop - vals["azurv1_growth_20mft"]) < 0.15
    balance_ok(o)


def test_config2_causality_and_balance():
    """P8: v = 1 pulse at x = 10 -> bins outside the light cone are exactly zero. P7 balance."""
    N = 50_000
    o = Oracle(mi.config2(n_hist=N)).run()
    T = o.tally(0)[:, 0, 0, 0, :]                    # [t, x]
    xe = np.array([j * 0.1 for j in range(201)]); te = np.array([j * 0.2 for j in range(101)])
    near = np.minimum(np.abs(xe[:-1] - 10.0), np.abs(xe[1:] - 10.0))
    outside = near[None, :] > te[1:, None] + 1e-12
    assert outside.sum() > 1000
    assert np.all(T[outside] == 0.0)
    inside = (near[None, :] + 0.1 < te[:-1, None]) & (te[:-1, None] < 3.0)
    assert np.all(T[inside] > 0.0)
    assert abs(T.sum() * N - 0) > 0
    balance_ok(o)
    assert o.counters()["census"] + o.counters()["leaks"] + o.counters()["captures"] == N


def test_config2_collision_estimator_agrees():
    """P9: per region, sum(flux) * Sigma_t ~ collisions in that region (collision estimator)."""
    N = 100_000
    # same physics, tally mesh = the 4 regions, so each bin is one region
    cfg = mi.config2(n_hist=N, nx_tally=4, nt_tally=1)
    o = Oracle(cfg).run()
    flux = o.tally(0).ravel() * N                    # raw track length per region
    st = np.array([1.0, 0.5, 2.0, 1.0])
    total_coll = o.counters()["collisions"]
    est = (flux * st).sum()
    # collisions ~ Poisson-like with mean est; 4 sigma with a factor for correlation
    assert abs(est - total_coll) < 4 * math.sqrt(total_coll) * 1.5


def test_tally_mesh_invariance():
    """P15: the tally mesh never creates events: counters (except segments) and the total are unchanged."""
    N = 20_000
    a = Oracle(mi.config2(n_hist=N)).run()
    b = Oracle(mi.config2(n_hist=N, nx_tally=1, nt_tally=1)).run()
    ca, cb = a.counters(), b.counters()
    for k in ca:
        if k != "segments":
            assert ca[k] == cb[k], k
    assert ca["segments"] > cb["segments"]
    sa, sb = a.tally(0).sum(), b.tally(0).sum()
    assert abs(sa - sb) <= 1e-12 * sb


@pytest.mark.parametrize("m", [0, 1])
def test_multigroup_infinite_medium_linear_solve(m):
    """P10: group fluxes of an infinite medium solve (diag St - Ss^T - chi (nu Sf)^T) phi = s."""
    mats, _ = mi.seeded_materials(2, fissile=(0,))
    G = 7
    s = mats["chi"][0].copy()
    St, Ss = mats["sigma_t"][m], mats["sigma_s"][m]
    nSf, chi = mats["nu"][m] * mats["sigma_f"][m], mats["chi"][m]
    A = np.diag(St) - Ss.T - np.outer(chi, nSf)
    phi = np.linalg.solve(A, s)
    assert np.all(phi > 0)                            # subcritical: the fixed-source problem is well posed
    N = 200_000
    o = Oracle(mi.infinite_multigroup(mats, m, s, n_hist=N, n_batch=10)).run(n_hist_per_batch=N // 10)
    got = o.tally(0).ravel()
    se = o.tally(1).ravel()
    assert np.all(se > 0)
    z = (got - phi) / se
    assert np.all(np.abs(z) < 4.5), z
    assert abs(got.sum() - phi.sum()) < 4 * np.sqrt((se ** 2).sum()) * 1.5
    balance_ok(o)


def test_config4_symmetry_and_no_leak():
    """P11: reflective lattice of identical pins: no leaks; pin-cell fluxes equal within statistics;
    the 3x3 sub-bin pattern has the square's symmetry."""
    N = 400_000
    o = Oracle(mi.config4(n_hist=N // 10, n_batch=10)).run()
    for b in range(10):
        assert o.counters(b)["leaks"] == 0
        balance_ok(o, b)
    T = o.tally(0).sum(axis=(0, 1, 2))                # [y, x] 51x51
    cells = T.reshape(17, 3, 17, 3).transpose(0, 2, 1, 3)   # [iy, ix, sy, sx]
    per_pin = cells.sum(axis=(2, 3))
    rel = per_pin.std() / per_pin.mean()
    assert rel < 0.04
    sub = cells.mean(axis=(0, 1))                     # 3x3 average pattern
    corners = sub[[0, 0, 2, 2], [0, 2, 0, 2]]; edges = sub[[0, 1, 1, 2], [1, 0, 2, 1]]
    assert corners.std() / corners.mean() < 0.02 and edges.std() / edges.mean() < 0.02
    assert not np.isclose(sub[1, 1], corners.mean(), rtol=0.02)   # fuel centre differs from moderator corners


def test_config5_small_balance_and_symmetric_source():
    """P7 on the voxel problem with census + comb (scaled down: 16^3 voxels, 5 steps)."""
    o = Oracle(mi.config5(n_hist=5000, n_batch=2, n_vox=16, n_steps=5, nusf_scale=1.0)).run()
    for b in range(2):
        balance_ok(o, b)
        assert o.counters(b)["leaks"] > 0
    assert o.counters(0)["fingerprint"] != o.counters(1)["fingerprint"]


@pytest.mark.slow
def test_one_over_sqrt_n_convergence():
    """P16: error vs the closed form falls like N^-1/2."""
    errs, Ns = [], [1000, 10_000, 100_000]
    for N in Ns:
        e = []
        for seed in range(8):
            o = Oracle(mi.config1(n_hist=N, seed=seed)).run()
            e.append(o.tally(0).item() - 2.0)
        errs.append(math.sqrt(np.mean(np.square(e))))
    slope = np.polyfit(np.log(Ns), np.log(errs), 1)[0]
    assert abs(slope + 0.5) < 0.15, (slope, errs)


def test_batches_are_independent_streams():
    """C.1: seed_b = seed + b, so batch 1 of seed 0 equals batch 0 of seed 1."""
    a = Oracle(mi.config1(n_hist=2000, n_batch=2, seed=0)).run()
    b = Oracle(mi.config1(n_hist=2000, n_batch=1, seed=1)).run()
    assert a.counters(1) == b.counters(0)
    assert a.tally(2).item() == b.tally(2).item()


def test_create_rejects_bad_input():
    cfg = mi.config1()
    cfg["materials"]["sigma_c"] = cfg["materials"]["sigma_c"] + 0.1      # Sigma_t mismatch
    with pytest.raises(ValueError):
        Oracle(cfg)
    cfg = mi.config2()
    cfg["tally"]["txs"] = cfg["tally"]["txs"][:-5]                      # mesh does not cover the slab
    with pytest.raises(ValueError):
        Oracle(cfg)
    cfg = mi.config3()
    cfg["census"]["t_census"] = cfg["census"]["t_census"] + 1e-9          # census time not a tally edge
    with pytest.raises(ValueError):
        Oracle(cfg)


def test_time_crossing_estimator():
    """Time-crossing estimator (DESIGN.md C.13): w*v of every particle alive when the
    time passes a tally time edge.  Infinite supercritical medium, edges every 0.05, census every 0.1:
    (a) closed form: the population at t is e^{alpha t} per source particle (4 sigma over batches), at
        edges crossed inside a flight and at edges that are census times alike;
    (b) exact: without a comb every weight is 1 and v = 1, so the census-edge bins ARE the census counts;
    (c) switching the block on changes no counter and no track-length bin."""
    import math
    edges = [0.05 * k for k in range(21)]
    cens = [0.1 * k for k in range(1, 11)]
    mk = lambda: mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, 1.0, t_edges=edges, t_census=cens,
                                    n_hist=20_000, n_batch=8)
    cfg = mk(); cfg["tally"]["time_crossing"] = 1
    o = Oracle(cfg).run()
    mean, se = o.tally(0), o.tally(1)
    assert mean.shape == (2, 20, 1, 1, 1, 1)
    for j in range(20):
        exact = math.exp(0.15 * edges[j + 1])
        assert abs(mean[1, j, 0, 0, 0, 0] - exact) <= 4.0 * se[1, j, 0, 0, 0, 0] + 1e-12, (j, mean[1, j].ravel(), exact)
    raw = o.tally(2)[1, :, 0, 0, 0, 0]
    for k in range(10):
        assert raw[2 * k + 1] == float(o.counters(7, k)["census"])
    p = Oracle(mk()).run()
    assert all(p.counters(b, k) == o.counters(b, k) for b in range(8) for k in range(10))
    assert np.array_equal(p.tally(2), o.tally(2)[0])


def test_time_crossing_causality_slab():
    """Config 2 (pulse at x = 10, v = 1): at time t_j nobody can be farther than t_j from the source."""
    cfg = mi.config2(n_hist=20_000); cfg["tally"]["time_crossing"] = 1
    o = Oracle(cfg).run()
    T = o.tally(2)[1, :, 0, 0, 0, :]                 # [time edge j+1][x bin]
    xs, ts = cfg["tally"]["txs"], cfg["tally"]["tts"]
    for j in range(T.shape[0]):
        far = np.minimum(np.abs(xs[:-1] - 10.0), np.abs(xs[1:] - 10.0)) > ts[j + 1]
        assert np.all(T[j, far] == 0.0)
    assert T.sum() > 0.0


# ---------------------------------------------------------------------------------------------
# k-eigenvalue mode (DESIGN.md §3 C.14), pins P18-P21
# ---------------------------------------------------------------------------------------------
def eig_balance_ok(o, N, batch=0):
    """Per generation: N in, every history ends in a capture, a fission or a leak; the fission bank
    (census counter) holds the secondaries; the generation estimate obeys k_c = k_{c-1} N_f / N
    exactly, computed here from the integer counters alone."""
    k = o.k_cycle(batch)
    k_prev = o.run_params_eig["k0"]
    for c in range(o.n_steps):
        cn = o.counters(batch, c)
        assert cn["lost"] == 0
        assert cn["captures"] + cn["fissions"] + cn["leaks"] == N
        assert cn["census"] == cn["secondaries"]
        assert cn["collisions"] == cn["scatters"] + cn["captures"] + cn["fissions"]
        assert k[c] == k_prev * float(cn["secondaries"]) / float(N)
        if c + 1 < o.n_steps:
            assert cn["comb_in"] == cn["census"] and cn["comb_out"] == N
        k_prev = k[c]


def run_eig(cfg):
    o = Oracle(cfg)
    o.run_params_eig = cfg["eigenvalue"]
    return o.run()


def test_eigenvalue_one_group_infinite_medium():
    """P18: k_inf = nu Sigma_f / Sigma_a = 0.75/0.6 = 1.25.  Every source neutron ends in a fission
    with probability p = Sigma_f/Sigma_a = 1/2 and then yields floor(nu/k + xi) children, so with the
    exact k each cycle estimate has mean k and variance <= k^2 (1/p - 1 + ...)/N: checked at 4 sigma
    from the cycle scatter AND against the a-priori bound.  Flux per source particle = 1/Sigma_a
    (mean track length to absorption, the parent dying at fission)."""
    N, I, A = 20_000, 5, 40
    cfg = mi.eigenvalue(mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, n_hist=N), I, A, k0=1.0)
    o = run_eig(cfg)
    k = o.k_cycle()[I:]
    assert abs(k.mean() - 1.25) < 4 * k.std(ddof=1) / math.sqrt(A)
    # a-priori: children per source neutron = B * n, B ~ Bernoulli(1/2), n in {2,3} (nu/k = 2):
    # var <= E[n^2]/2 - 1 <= 9/2 - 1; sigma of a cycle estimate <= 1.25 * sqrt(3.5/N)
    assert abs(k.mean() - 1.25) < 4 * 1.25 * math.sqrt(3.5 / (N * A)) * 1.5
    flux = o.tally(0).item()
    assert abs(flux - 1 / 0.6) < 4 * (1 / 0.6) / math.sqrt(N * A)
    assert o.counters(0, 0)["segments"] == 0 and o.counters(0, I)["segments"] > 0   # inactive cycles do not score
    eig_balance_ok(o, N)


def test_eigenvalue_is_independent_of_k0():
    """P18b: the converged k does not depend on the starting guess (the normalisation cancels)."""
    N = 20_000
    ks = []
    for k0 in (0.6, 1.25, 2.0):
        cfg = mi.eigenvalue(mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, n_hist=N), 3, 20, k0=k0)
        k = run_eig(cfg).k_cycle()[3:]
        ks.append((k.mean(), k.std(ddof=1) / math.sqrt(20)))
    for m, s in ks:
        assert abs(m - 1.25) < 4 * s + 1e-3


def test_eigenvalue_multigroup_infinite_medium_vs_numpy_eig():
    """P19: infinite homogeneous fuel of the config-4 set: k_inf and the group spectrum are the
    dominant eigenpair of the textbook multigroup balance
        (diag(Sigma_t) - Sigma_s^T) phi = (1/k) chi (nu Sigma_f)^T phi
    solved with numpy.linalg.eig (a library routine the oracle does not use)."""
    mats, _ = mi.seeded_materials(2, fissile=(0,), nusf_scale=7.0)
    m = 0
    st, ss = mats["sigma_t"][m], mats["sigma_s"][m]
    nusf, chi = mats["nu"][m] * mats["sigma_f"][m], mats["chi"][m]
    A_ = np.diag(st) - ss.T
    F = np.outer(chi, nusf)
    w, v = np.linalg.eig(np.linalg.solve(A_, F))
    i = int(np.argmax(w.real))
    k_ref = float(w[i].real)
    phi = np.abs(v[:, i].real)
    N, I, A = 20_000, 5, 30
    cfg = mi.eigenvalue(mi.infinite_multigroup(mats, m, chi, n_hist=N), I, A, k0=1.0)
    o = run_eig(cfg)
    k = o.k_cycle()[I:]
    assert abs(k.mean() - k_ref) < 4 * k.std(ddof=1) / math.sqrt(A) + 1e-4
    assert abs(k.mean() / k_ref - 1) < 0.01
    # spectrum: flux per source particle; normalise both to the production rate nuSf.phi = k
    flux = o.tally(0).reshape(-1)
    phi = phi * (k_ref / float(nusf @ phi))
    err = o.tally(1).reshape(-1)     # one batch: no batch error; use a 2 % band on groups that matter
    big = phi > 0.02 * phi.max()
    assert np.all(np.abs(flux[big] / phi[big] - 1) < 0.03), (flux, phi)
    eig_balance_ok(o, N)


def test_eigenvalue_leaking_slab_track_length_estimate_of_k():
    """P20: bare fissile slab (vacuum faces): no closed form for k, but two independent estimators
    of the same run must agree — the generation estimate (fission-bank size, comb normalisation) and
    the track-length estimate k_TL = sum_bins nu Sigma_f phi(bin) per source particle (tally path).
    Also: leakage makes k smaller than k_inf, and a wider slab leaks less."""
    N, I, A = 20_000, 5, 40
    out = []
    for width in (4.0, 12.0):
        cfg = mi.eigenvalue(mi.fissile_slab(width=width, n_hist=N), I, A, k0=1.0)
        o = run_eig(cfg)
        k = o.k_cycle()[I:]
        k_gen, s_gen = k.mean(), k.std(ddof=1) / math.sqrt(A)
        k_tl = float(o.tally(0).sum() * 2.5 * 0.2)
        # both carry statistical noise of the same order
        assert abs(k_tl - k_gen) < 4 * math.hypot(s_gen, s_gen) + 2e-3, (k_tl, k_gen, s_gen)
        c = o.counters(0, -1)
        assert c["leaks"] > 0
        eig_balance_ok(o, N)
        out.append(k_gen)
    k_inf = 2.5 * 0.2 / 0.5
    assert out[0] < out[1] < k_inf
    # symmetric problem: the converged flux is symmetric about the mid-plane (4 sigma, Poisson-like bound)
    f = o.tally(0).reshape(-1)
    assert np.all(np.abs(f - f[::-1]) < 0.05 * f.max())


def test_eigenvalue_rejects_time_dependent_and_bad_arguments():
    cfg = mi.config3(n_hist=100)
    cfg["eigenvalue"] = dict(n_inactive=1, n_active=1, k0=1.0)
    with pytest.raises(ValueError):
        Oracle(cfg)
    for bad in (dict(n_inactive=-1, n_active=1, k0=1.0), dict(n_inactive=0, n_active=0, k0=1.0),
                dict(n_inactive=0, n_active=1, k0=0.0)):
        cfg = mi.config1(n_hist=100)
        cfg["eigenvalue"] = bad
        with pytest.raises(ValueError):
            Oracle(cfg)


# ---------------------------------------------------------------------------------------------
# implicit capture, weight roulette, weighted comb (DESIGN.md §3 C.15), pins P22-P25
# ---------------------------------------------------------------------------------------------
def test_implicit_capture_infinite_medium_flux_with_roulette():
    """P22: implicit capture + roulette are unbiased: the config-1 flux stays S/Sigma_a = 2 (4 sigma of
    the batch standard error).  Every history ends in the roulette (captures = N): nothing else can end
    it in an infinite medium without a time cut-off.  The roulette must be played BELOW w_roulette only:
    with w_survive = 0.5 and c = 0.5 the first collision (w = 0.5) is not rouletted at w_roulette = 0.5
    but the second is, so collisions per history >= 2."""
    N, B = 20_000, 10
    o = Oracle(mi.implicit_capture(mi.config1(n_hist=N, n_batch=B), 0.5, 0.5)).run()
    flux, se = float(o.tally(0).ravel()[0]), float(o.tally(1).ravel()[0])
    assert se > 0 and abs(flux - 2.0) < 4 * se, (flux, se)
    # implicit capture reduces the variance of the analog estimate (analog: Var = 4/ (N B) per particle)
    assert se < math.sqrt(4.0 / (N * B))
    for b in range(B):
        c = o.counters(b)
        assert c["captures"] == N and c["fissions"] == 0 and c["census"] == 0
        assert c["collisions"] == c["scatters"] + c["captures"]
        assert c["collisions"] >= 2 * N


def test_implicit_capture_time_dependent_no_roulette():
    """P23: without the roulette nobody dies before the census: census = N exactly, no captures, and
    the flux over [0, T] is (1 - e^{-Sigma_a v T}) / Sigma_a.  The weight that reaches the census is
    e^{-Sigma_a v T} per source particle: checked through the time-crossing block, which scores w v at
    t = T."""
    N, B, T = 20_000, 8, 3.0
    cfg = mi.infinite_medium(1.0, 0.5, 0.5, 0.0, 0.0, 1.0, t_edges=[0.0, T], t_census=[T], n_hist=N, n_batch=B)
    cfg["tally"]["time_crossing"] = 1
    o = Oracle(mi.implicit_capture(cfg, 0.0, 1.0)).run()
    mean, se = o.tally(0).reshape(2, -1), o.tally(1).reshape(2, -1)
    assert abs(mean[0, 0] - (1 - math.exp(-0.5 * T)) / 0.5) < 4 * se[0, 0]
    assert abs(mean[1, 0] - math.exp(-0.5 * T)) < 4 * se[1, 0]
    for b in range(B):
        c = o.counters(b)
        assert c["census"] == N and c["captures"] == 0 and c["collisions"] == c["scatters"]


def test_implicit_capture_leaves_slab_expectations_unchanged():
    """P24: analog and implicit-capture runs of config 2 (different histories, same expectations):
    region-integrated fluxes agree within 4 combined sigma; leaks + census + captures = N in both."""
    N, B = 20_000, 8
    a = Oracle(mi.config2(n_hist=N, n_batch=B, nx_tally=4, nt_tally=2)).run()
    i = Oracle(mi.implicit_capture(mi.config2(n_hist=N, n_batch=B, nx_tally=4, nt_tally=2), 0.1, 0.3)).run()
    ma, sa, mi_, si = a.tally(0).ravel(), a.tally(1).ravel(), i.tally(0).ravel(), i.tally(1).ravel()
    assert np.all(np.abs(ma - mi_) < 4 * np.hypot(sa, si)), (ma - mi_) / np.hypot(sa, si)
    for o in (a, i):
        c = o.counters(0)
        assert c["leaks"] + c["census"] + c["captures"] == N
    assert i.counters(0)["captures"] < a.counters(0)["captures"]


def test_weighted_comb_unit():
    """P25: the weighted comb's teeth, checked against exact rational arithmetic: tooth j sits at
    (j + a) W_q / M on the axis of cumulated fixed-point weights and takes the entry whose interval
    [P_i, P_{i+1}) holds it.  Zero-weight entries are never taken, indices are monotone, entry i is
    taken floor or ceil of q_i M / W_q times, all survivors weigh W / M, and equal weights give the
    uniform comb's indices."""
    from fractions import Fraction
    import ctypes as C
    from oracle.binding import lib
    L = lib()
    rng = np.random.default_rng(7)
    for N, M in ((1000, 777), (500, 2000), (1, 5), (4096, 4096)):
        w = rng.random(N) ** 3 * 2.0
        w[rng.random(N) < 0.1] = 0.0
        if N == 1:
            w[0] = 0.37
        a = float(rng.random())
        idx = np.zeros(M, np.uint64)
        w_out = C.c_double()
        assert L.oracle_comb_weighted(N, M, a, w.ctypes.data_as(C.POINTER(C.c_double)),
                                      idx.ctypes.data_as(C.POINTER(C.c_uint64)), C.byref(w_out)) == 0
        q = [int(Fraction(float(x)) * 2**32 + Fraction(1, 2)) for x in w]
        P = np.concatenate([[0], np.cumsum(np.array(q, dtype=object))])
        Wq = int(P[-1])
        assert w_out.value == (Wq / 2**32) / M
        idx = idx.astype(np.int64)
        assert np.all(np.diff(idx) >= 0)
        assert all(q[i] > 0 for i in idx)
        exact_mismatch = 0
        for j in range(M):
            t = (Fraction(j) + Fraction(a)) * Fraction(Wq, M)
            t = min(int(t), Wq - 1)
            i = int(np.searchsorted(np.array(P[1:], dtype=object), t, side="right"))
            exact_mismatch += int(i != idx[j])
            assert abs(i - idx[j]) <= 1 or q[min(i, idx[j]) + 1] == 0
        assert exact_mismatch <= max(1, M // 1000)      # (the oracle's tooth position is one binary64 product)
        counts = np.bincount(idx, minlength=N)
        for i in range(N):
            m = Fraction(q[i] * M, Wq)
            assert math.floor(m) - (1 if exact_mismatch else 0) <= counts[i] <= math.ceil(m) + (1 if exact_mismatch else 0)
    # equal weights: the uniform comb
    N, M, a = 3000, 1234, 0.31415
    w = np.full(N, 0.75)
    idx = np.zeros(M, np.uint64); ref = np.zeros(M, np.uint64); w_out = C.c_double()
    L.oracle_comb_weighted(N, M, a, w.ctypes.data_as(C.POINTER(C.c_double)), idx.ctypes.data_as(C.POINTER(C.c_uint64)), C.byref(w_out))
    L.oracle_comb_indices(N, M, C.c_double(a), ref.ctypes.data_as(C.POINTER(C.c_uint64)))
    assert np.count_nonzero(idx != ref) <= 1 and w_out.value == 0.75 * N / M
    # a negative or huge weight is refused
    bad = np.array([1.0, -1.0])
    assert L.oracle_comb_weighted(2, 2, 0.5, bad.ctypes.data_as(C.POINTER(C.c_double)), idx.ctypes.data_as(C.POINTER(C.c_uint64)), C.byref(w_out)) == 1


@pytest.mark.parametrize("roulette", [(0.0, 1.0), (0.4, 0.8)])
def test_config3_growth_with_implicit_capture_and_weighted_comb(roulette):
    """P26: config 3 with implicit capture and the weighted comb at every census still grows as
    e^{alpha t}: interval fluxes (e^{a t_k} - e^{a t_{k-1}})/a within 4 sigma (same bound as P5, whose
    analog variance is an upper bound here); the comb keeps the population at M."""
    N = 100_000
    o = Oracle(mi.implicit_capture(mi.config3(n_hist=N), *roulette)).run()
    a = 0.15
    tk = np.array([0.1 * k for k in range(21)])
    expect = (np.exp(a * tk[1:]) - np.exp(a * tk[:-1])) / a
    got = o.tally(0).ravel()
    tol = 4 * expect * np.sqrt((0.5 + 2.0 * tk[1:]) / N)
    assert np.all(np.abs(got - expect) < tol), (got - expect) / tol
    assert all(o.counters(0, k)["comb_out"] == N for k in range(19))
    # the population in PARTICLES grows faster than e^{alpha t} (nobody is captured): nu Sigma_f v dt per step
    assert o.counters(0, 5)["comb_in"] / N > math.exp(0.015) + 0.02


def test_implicit_capture_rejects_bad_arguments():
    for bad in ((-1.0, 1.0), (0.5, 0.25), (0.1, 1e9)):
        with pytest.raises(ValueError):
            Oracle(mi.implicit_capture(mi.config1(n_hist=10), *bad))
    cfg = mi.eigenvalue(mi.implicit_capture(mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, n_hist=10)), 1, 1)
    with pytest.raises(ValueError):
        Oracle(cfg)


# ---------------------------------------------------------------------------------------------
# delayed neutrons (DESIGN.md §3 C.16), pins P27-P30
# ---------------------------------------------------------------------------------------------
def _point_kinetics_interval_flux(st, sc, sf, nu, nud, lam, tk):
    """Infinite homogeneous 1-group medium, v = 1, J precursor groups: the exact point-kinetics
    equations  n' = ((nu - sum nud) sf - (sc + sf)) n + sum lam_j C_j,  C_j' = nud_j sf n - lam_j C_j,
    n(0) = 1, C(0) = 0.  Returns int_{t_k}^{t_{k+1}} n dt from the matrix exponential (scipy)."""
    from scipy.linalg import expm
    nud, lam = np.atleast_1d(nud), np.atleast_1d(lam)
    J = len(nud)
    B = np.zeros((J + 2, J + 2))
    B[0, 0] = (nu - nud.sum()) * sf - (sc + sf)
    B[0, 1:J + 1] = lam
    for j in range(J):
        B[1 + j, 0] = nud[j] * sf
        B[1 + j, 1 + j] = -lam[j]
    B[J + 1, 0] = 1.0                                  # running integral of n
    y0 = np.zeros(J + 2); y0[0] = 1.0
    I = np.array([(expm(B * t) @ y0)[J + 1] for t in tk])
    return np.diff(I)


@pytest.mark.parametrize("comb", [0, 1])
def test_delayed_neutrons_point_kinetics(comb):
    """P27: with a large delayed fraction (nu_d = 0.6 + 0.3 of nu = 2.4) and decay constants of the
    order of the census interval the flux history differs strongly from the all-prompt one (the
    medium is prompt-subcritical and exactly critical with the delayed neutrons) and must follow the exact
    point-kinetics solution in every census interval (4 sigma of the batch error); with and without
    the comb (waiting precursors are combed with the neutrons)."""
    st, ss, sc, sf, nu = 1.0, 0.4, 0.35, 0.25, 2.4
    nud, lam = [0.6, 0.3], [0.8, 3.0]
    tk = np.linspace(0.0, 4.0, 9)
    N, B = 20_000, 10
    cfg = mi.infinite_medium(st, ss, sc, sf, nu, 1.0, t_edges=tk, t_census=tk[1:], comb_target=N if comb else 0,
                             n_hist=N, n_batch=B)
    o = Oracle(mi.delayed(cfg, [[nud]], [lam])).run()
    expect = _point_kinetics_interval_flux(st, sc, sf, nu, nud, lam, tk)
    got, se = o.tally(0).ravel(), o.tally(1).ravel()
    assert np.all(np.abs(got - expect) < 4 * se), (got - expect) / se
    # the all-prompt medium with the same total nu has alpha = nu sf - sa = 0: flux 0.5 per interval
    assert abs(expect[-1] - 0.5) > 20 * se[-1]
    c = o.counters(0)
    assert c["flights"] - c["segments"] > 0            # waiting precursors: census events of length 0
    if not comb:
        balance_ok(o)


def test_delayed_neutrons_do_not_change_time_integrated_flux():
    """P28: time-independent, subcritical: the total flux is 1/(Sigma_a - nu Sigma_f) whatever part of
    nu is delayed (a delay moves a neutron in time only)."""
    N, B = 20_000, 10
    cfg = mi.infinite_medium(1.0, 0.4, 0.4, 0.2, 2.0, n_hist=N, n_batch=B)
    o = Oracle(mi.delayed(cfg, [[[0.5, 0.2]]], [[0.1, 2.0]])).run()
    got, se = float(o.tally(0).ravel()[0]), float(o.tally(1).ravel()[0])
    assert abs(got - 1.0 / (0.6 - 0.4)) < 4 * se
    balance_ok(o)


def test_delayed_spectrum_multigroup_linear_solve():
    """P29: 7 groups, delayed neutrons with their own (softer) spectra: the time-integrated group
    fluxes solve (diag St - Ss^T - chi_p (nu_p Sf)^T - sum_j chi_d,j (nu_d,j Sf)^T) phi = s.  The
    solution differs from the all-prompt one by many sigma, so a wrong spectrum or yield fails."""
    mats, _ = mi.seeded_materials(2, fissile=(0,))
    m, G, J = 0, 7, 3
    s = mats["chi"][0].copy()
    cfg = mi.seeded_delayed(mi.infinite_multigroup(mats, m, s, n_hist=20_000, n_batch=10), J=J, beta=0.4)
    d = cfg["delayed"]
    St, Ss, Sf, nu, chi = (cfg["materials"][k][0] for k in ("sigma_t", "sigma_s", "sigma_f", "nu", "chi"))
    nud = d["nu_delayed"][0]                           # [G][J]
    A = np.diag(St) - Ss.T - np.outer(chi, (nu - nud.sum(axis=1)) * Sf)
    for j in range(J):
        A -= np.outer(d["chi_delayed"][0, j], nud[:, j] * Sf)
    phi = np.linalg.solve(A, s)
    phi_prompt = np.linalg.solve(np.diag(St) - Ss.T - np.outer(chi, nu * Sf), s)
    o = Oracle(cfg).run()
    got, se = o.tally(0).ravel(), o.tally(1).ravel()
    assert np.all(np.abs(got - phi) < 4.5 * se), (got - phi) / se
    assert np.max(np.abs(phi_prompt - phi) / se) > 10
    balance_ok(o)


def test_delayed_neutrons_eigenvalue_and_bad_arguments():
    """P30: k_inf = nu Sigma_f / Sigma_a does not depend on the delayed split (1 group).  Bad data
    (sum of delayed yields above nu, a decay constant <= 0, a spectrum that does not sum to 1) refused."""
    N, I, A = 20_000, 3, 20
    base = mi.infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, n_hist=N)
    o = run_eig(mi.eigenvalue(mi.delayed(base, [[[0.4, 0.3]]], [[0.5, 2.0]]), I, A))
    k = o.k_cycle()[I:]
    assert abs(k.mean() - 1.25) < 4 * k.std(ddof=1) / math.sqrt(A) + 1e-3
    for nud, lam, chd in (([[[2.0, 1.0]]], [[0.5, 2.0]], None), ([[[0.4, 0.3]]], [[0.5, 0.0]], None),
                          ([[[0.4, 0.3]]], [[0.5, 2.0]], [[[0.9], [1.0]]])):
        with pytest.raises(ValueError):
            Oracle(mi.delayed(base, nud, lam, chd))


# ---------------------------------------------------------------------------------------------
# source with a time extent (DESIGN.md §3 C.17), pin P31
# ---------------------------------------------------------------------------------------------
def test_source_window_closed_form():
    """P31: infinite 1-group medium, Sigma_a v = a = 0.5, unit source spread uniformly over [0, 2]:
    n' = S(t) - a n gives n(t) = (1 - e^{-a t})/(2a) for t <= 2 and n(2) e^{-a (t-2)} afterwards; the
    flux of every census interval is the integral of n (4 batch-sigma).  Census times cut the window, so
    source particles born after a census wait in the census bank (census events of length 0); a pulse at
    t = 0 instead of the window (the default) is > 20 sigma away."""
    a, T = 0.5, 2.0
    tk = np.linspace(0.0, 4.0, 9)
    N, B = 20_000, 10
    cfg = mi.infinite_medium(1.0, 0.5, 0.5, 0.0, 0.0, 1.0, t_edges=tk, t_census=tk[1:], n_hist=N, n_batch=B)
    cfg["source"]["t_end"] = T

    def integral(t):
        n2 = (1 - math.exp(-a * T)) / (T * a)
        i2 = (T - (1 - math.exp(-a * T)) / a) / (T * a)
        return (t - (1 - math.exp(-a * t)) / a) / (T * a) if t <= T else i2 + n2 * (1 - math.exp(-a * (t - T))) / a

    expect = np.diff([integral(t) for t in tk])
    o = Oracle(cfg).run()
    got, se = o.tally(0).ravel(), o.tally(1).ravel()
    assert np.all(np.abs(got - expect) < 4 * se), (got - expect) / se
    pulse = np.diff([(1 - math.exp(-a * t)) / a for t in tk])
    assert abs(pulse[0] - expect[0]) > 20 * se[0]
    c = o.counters(0)
    assert c["flights"] - c["segments"] > N // 2          # waiting source particles
    assert c["source"] == N and c["captures"] + o.counters(0, 7)["census"] == N
    with pytest.raises(ValueError):
        bad = mi.infinite_medium(n_hist=10); bad["source"]["t_end"] = 0.0
        Oracle(bad)


# ---------------------------------------------------------------------------------------------
# geometry of configs 4 and 5 with ONE material everywhere: every surface must be transparent (P32)
# ---------------------------------------------------------------------------------------------
def _moderator_spectrum(mats, m, s):
    St, Ss = mats["sigma_t"][m], mats["sigma_s"][m]
    return np.linalg.solve(np.diag(St) - Ss.T, s)


def test_config4_geometry_is_transparent_for_one_material():
    """P32a: the 17 x 17 reflective pin lattice of config 4 with the moderator inside the pins too and
    no time cut-off is an infinite homogeneous medium: the group fluxes must solve (diag St - Ss^T) phi
    = s (numpy.linalg.solve) although every history crosses cylinders and lattice planes and reflects
    off the box faces; no leaks; the flux is flat over the 17 x 17 cells apart from the source being
    inside the pins (cell integrals equal within noise, by symmetry of pin and moderator)."""
    N, B = 10_000, 10
    cfg = mi.config4(n_hist=N, n_batch=B)
    cfg["geometry"] = dict(cfg["geometry"]); cfg["geometry"]["mat_inner"] = np.ones((1, 17, 17), np.int32)
    cfg["tally"] = dict(cfg["tally"]); cfg["tally"]["tts"] = np.array([0.0, mi.INF])
    cfg["census"] = dict(t_census=np.zeros(0), comb_target=0)
    o = Oracle(cfg).run()
    s = cfg["source"]["group_pdf"]
    phi = _moderator_spectrum(cfg["materials"], 1, s)
    mean, se = o.tally(0)[0], o.tally(1)[0]            # [g][z][y][x]
    got = mean.sum(axis=(1, 2, 3))
    # the bins of one group are correlated; bound the error of the sum by the sum of the bin errors
    tol = 4.5 * np.sqrt((se ** 2).sum(axis=(1, 2, 3))) * 3.0
    assert np.all(np.abs(got - phi) < tol), (got - phi) / tol
    assert np.all(np.abs(got - phi) < 0.03 * phi)
    c = o.counters(0)
    assert c["leaks"] == 0 and c["reflections"] > 0 and c["crossings"] > N and c["captures"] == N
    cells = mean.sum(axis=(0, 1)).reshape(17, 3, 17, 3).sum(axis=(1, 3))
    assert cells.std() / cells.mean() < 0.05


def test_config5_geometry_is_transparent_for_one_material():
    """P32b: config 5's voxel lattice (16^3 here) filled with one non-fissile material, reflective
    faces, no census: again the infinite-medium spectrum, through several voxel crossings and
    reflections per history, and a flat flux over the voxels."""
    N, B = 5_000, 10
    cfg = mi.config5(n_hist=N, n_batch=B, n_vox=16, n_steps=1, nusf_scale=1.0)
    g = dict(cfg["geometry"]); g["mat_outer"] = np.full((16, 16, 16), 5, np.int32); g["bc"] = np.ones(6, np.int32)
    cfg["geometry"] = g
    cfg["tally"] = dict(cfg["tally"]); cfg["tally"]["tts"] = np.array([0.0, mi.INF])
    cfg["census"] = dict(t_census=np.zeros(0), comb_target=0)
    o = Oracle(cfg).run()
    s = cfg["source"]["group_pdf"]
    phi = _moderator_spectrum(cfg["materials"], 5, s)
    mean, se = o.tally(0)[0], o.tally(1)[0]
    got = mean.sum(axis=(1, 2, 3))
    tol = 4.5 * np.sqrt((se ** 2).sum(axis=(1, 2, 3))) * 3.0
    assert np.all(np.abs(got - phi) < tol), (got - phi) / tol
    assert np.all(np.abs(got - phi) < 0.03 * phi)
    c = o.counters(0)
    assert c["leaks"] == 0 and c["reflections"] > 0 and c["crossings"] > 3 * N and c["captures"] == N
    vox = mean.sum(axis=0)
    assert abs(vox[:8].sum() - vox[8:].sum()) < 0.02 * vox.sum()
    assert abs(vox[:, :8].sum() - vox[:, 8:].sum()) < 0.02 * vox.sum()
    assert abs(vox[:, :, :8].sum() - vox[:, :, 8:].sum()) < 0.02 * vox.sum()


# ---------------------------------------------------------------------------------------------
# P33: the direction law (C.4) — used by the source, every scatter and every fission child.
# Infinite-medium pins are direction-blind and symmetric geometries hide any angular law, so it is
# pinned on its own: exact unit vectors, the moments of the uniform distribution on the sphere by
# quadrature over the two uniforms, and the leakage of a purely absorbing slab with the source OFF
# centre, 1/2 [E2(a) + E2(b)], with the slab normal along x, then y, then z.
def _iso(a, b):
    import ctypes as C
    from oracle import lib
    u = (C.c_double * 3)()
    lib().oracle_isotropic(float(a), float(b), u)
    return np.array([u[0], u[1], u[2]])


def test_isotropic_direction_is_a_unit_vector_with_sphere_moments():
    rng = np.random.default_rng(33)
    for a, b in rng.random((2000, 2)):
        u = _iso(a, b)
        assert abs(float(np.dot(u, u)) - 1.0) <= 4 * 2.0 ** -52
    # the extreme uniforms the generator can produce, (k + 1/2) 2^-52 at k = 0 and k = 2^52 - 1
    for a in (2.0 ** -53, 1.0 - 2.0 ** -53, 0.5):
        for b in (2.0 ** -53, 0.25, 0.5, 0.75, 1.0 - 2.0 ** -53):
            u = _iso(a, b)
            assert np.all(np.isfinite(u)) and abs(float(np.dot(u, u)) - 1.0) <= 4 * 2.0 ** -52
    # midpoint quadrature over (a, b) in (0,1)^2: E[u] = 0, E[u_i u_j] = delta_ij / 3, E[u_i^4] = 1/5,
    # E[|u_i|] = 1/2; P(u_i > 1/2) = 1/4 (each component is uniform on [-1, 1]: Archimedes)
    n = 400
    g = (np.arange(n) + 0.5) / n
    U = np.array([[_iso(a, b) for b in g] for a in g]).reshape(-1, 3)
    assert np.all(np.abs(U.mean(axis=0)) < 1e-12)
    second = U.T @ U / len(U)
    assert np.all(np.abs(second - np.eye(3) / 3.0) < 2e-5), second
    assert np.all(np.abs((U ** 4).mean(axis=0) - 0.2) < 2e-5)
    assert np.all(np.abs(np.abs(U).mean(axis=0) - 0.5) < 2e-3)
    for i in range(3):
        assert abs(np.mean(U[:, i] > 0.5) - 0.25) < 5e-3
        assert abs(np.mean(U[:, i] < -0.5) - 0.25) < 5e-3
    # mu = 2 a - 1 sits on the x axis (S8); phi runs over the whole turn, counter-clockwise from +y
    assert _iso(0.75, 0.3)[0] == 0.5 and _iso(0.25, 0.3)[0] == -0.5
    q = math.sqrt(0.75)
    assert np.allclose(_iso(0.75, 0.125), [0.5, q * math.sqrt(0.5), q * math.sqrt(0.5)], rtol=0, atol=1e-15)
    assert np.allclose(_iso(0.75, 0.625), [0.5, -q * math.sqrt(0.5), -q * math.sqrt(0.5)], rtol=0, atol=1e-15)
    assert np.allclose(_iso(0.75, 0.375), [0.5, -q * math.sqrt(0.5), q * math.sqrt(0.5)], rtol=0, atol=1e-15)


def _absorbing_plate(axis, lo, hi, n_hist, seed):
    """One purely absorbing cell (Sigma_t = 1), finite along `axis` only, vacuum faces, isotropic
    point source at the origin."""
    cfg = mi.infinite_medium(1.0, 0.0, 1.0, n_hist=n_hist, seed=seed)
    key = ("xs", "ys", "zs")[axis]
    cfg["geometry"][key] = np.array([lo, hi])
    cfg["tally"]["t" + key] = np.array([lo, hi])
    cfg["name"] = "absorbing_plate_" + key
    return cfg


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_isotropic_source_slab_leakage_is_E2(axis):
    """A particle with direction cosine c to the slab normal leaks through the face at distance h with
    probability exp(-h / |c|); c uniform on [-1, 1] gives 1/2 E2(a) towards -a and 1/2 E2(b) towards +b.
    a != b, so a one-sided or half-turn angular law fails; three (a, b) pairs sample the distribution of
    |c| at different depths."""
    from scipy.special import expn
    N = 200_000
    for a, b in ((0.5, 2.0), (1.0, 0.25), (2.0, 1.0)):
        o = Oracle(_absorbing_plate(axis, -a, b, N, seed=7 + axis)).run()
        c = o.counters()
        p = 0.5 * (expn(2, a) + expn(2, b))
        assert c["captures"] + c["leaks"] == N and c["scatters"] == 0
        assert abs(c["leaks"] / N - p) < 4 * math.sqrt(p * (1 - p) / N), (axis, a, b, c["leaks"] / N, p)
        # track length per history: 1 - leak probability (every history ends in a capture or a leak and
        # the mean chord to a capture at Sigma_t = 1 obeys <l> = P(capture)/Sigma_t)
        assert abs(o.tally(0).item() - (1 - p)) < 4 * math.sqrt(1.0 / N)
        o.close()


# ---------------------------------------------------------------------------------------------
# P34: which material is inside the pin.  One cell with a purely absorbing pin (mat_inner) in a void
# (mat_outer, Sigma_t = 1e-9), vacuum faces, source uniform inside the pin (kind 2): the leakage is the
# first-flight escape probability of an infinite cylinder,
#   P = 1/(pi R^2) int_0^R 2 pi r dr  1/(2 pi) int_0^2pi dphi  Ki2(Sigma l(r, phi)),
#   l = -r cos phi + sqrt(R^2 - r^2 sin^2 phi),  Ki2(x) = int_0^pi/2 sin(th) exp(-x / sin th) dth,
# evaluated here by quadrature.  With mat_inner and mat_outer swapped nothing is absorbed (leak = 1);
# a wrong radius, a non-uniform source in the disc or a wrong cylinder root all move it.
def _cylinder_escape(sig_r):
    n = 400
    th = (np.arange(n) + 0.5) / n * (math.pi / 2)

    def ki2(x):
        return np.sum(np.sin(th)[None, :] * np.exp(-x[:, None] / np.sin(th)[None, :]), axis=1) * (math.pi / 2 / n)

    m = 300
    r = np.sqrt((np.arange(m) + 0.5) / m)                  # equal-area radii (R = 1)
    ph = (np.arange(m) + 0.5) / m * 2 * math.pi
    rr, pp = np.meshgrid(r, ph, indexing="ij")
    ell = -rr * np.cos(pp) + np.sqrt(1.0 - (rr * np.sin(pp)) ** 2)
    return float(ki2(sig_r * ell.ravel()).mean())


@pytest.mark.parametrize("sigma,R", [(1.0, 0.54), (4.0, 0.54), (2.0, 0.3)])
def test_pin_material_is_inside_the_cylinder_escape_probability(sigma, R):
    N = 200_000
    mats = mi._materials_1g([sigma, 1e-9], [0.0, 0.0], [sigma, 1e-9], [0.0, 0.0], [0.0, 0.0])
    geom = dict(xs=np.array([0.0, 1.26]), ys=np.array([0.0, 1.26]), zs=np.array([-mi.INF, mi.INF]),
                mat_outer=np.full((1, 1, 1), 1, np.int32), mat_inner=np.full((1, 1, 1), 0, np.int32),
                radius=np.full((1, 1, 1), R), bc=np.zeros(6, np.int32))
    pdf = np.ones(1)
    cfg = dict(name="pin_escape", materials=mats, geometry=geom,
               source=dict(kind=2, lo=np.zeros(3), hi=np.zeros(3), isotropic=1, dir=np.array([1.0, 0.0, 0.0]),
                           group_pdf=pdf, t0=0.0),
               tally=dict(txs=geom["xs"].copy(), tys=geom["ys"].copy(), tzs=geom["zs"].copy(), tts=np.array([0.0, mi.INF])),
               census=dict(t_census=np.zeros(0), comb_target=0),
               run=dict(seed=11, n_hist_per_batch=N, n_batch=1))
    o = Oracle(cfg).run()
    c = o.counters()
    p = _cylinder_escape(sigma * R)
    # (the void absorbs 1e-9 per cm: < 1e-8 of the leakers)
    assert abs(c["leaks"] / N - p) < 4 * math.sqrt(p * (1 - p) / N) + 1e-7, (c["leaks"] / N, p)
    assert c["crossings"] == c["leaks"] + (c["captures"] - (N - c["leaks"]))  # one cylinder crossing per escaping particle
    # sanity of the quadrature against the two limits of the escape probability
    assert abs(_cylinder_escape(1e-6) - 1.0) < 1e-5 and abs(_cylinder_escape(200.0) - 1.0 / (2 * 200.0)) < 2e-4
    o.close()
