"""Pins of the quadric-surface CSG (DESIGN.md section 3 C.18) and of moving surfaces (C.19) in the oracle:
root residuals and brute force for the surface distance, closed-form escape probabilities of a sphere
and of a (tilted) cylinder, the slab of config 2 rebuilt from quadric planes, and the exact attenuation
behind a moving interface."""
import ctypes as C
import math

import numpy as np
import pytest

import mcdc_inputs as mi
from oracle import Oracle, lib

INF = float("inf")


def qdist(q, sense, r, u):
    qq = np.ascontiguousarray(q, dtype=np.float64)
    return lib().oracle_quadric_distance(qq.ctypes.data_as(C.POINTER(C.c_double)), float(sense), *map(float, r), *map(float, u))


def feval(q, r):
    x, y, z = r
    return (q[0] * x * x + q[1] * y * y + q[2] * z * z + q[3] * x * y + q[4] * y * z + q[5] * z * x +
            q[6] * x + q[7] * y + q[8] * z + q[9])


def random_quadrics(rng):
    R = np.linalg.qr(rng.normal(size=(3, 3)))[0]
    c = rng.uniform(-1, 1, 3)

    def gen(diag, k):
        M = R @ np.diag(diag) @ R.T
        return mi.quadric_general(M, -2 * M @ c, c @ M @ c + k)
    return {
        "sphere": mi.quadric_sphere(c, rng.uniform(0.5, 2)),
        "ellipsoid": gen(rng.uniform(0.3, 2, 3), -1.0),
        "cylinder": mi.quadric_cylinder(c, rng.normal(size=3), rng.uniform(0.3, 1.5)),
        "cone": gen([1.0, 1.0, -rng.uniform(0.3, 2)], 0.0),
        "hyperboloid1": gen([1.0, rng.uniform(0.5, 2), -1.0], -1.0),
        "hyperboloid2": gen([1.0, rng.uniform(0.5, 2), -1.0], 1.0),
        "paraboloid": mi.quadric_general(np.diag([1.0, rng.uniform(0.5, 2), 0.0]), [0, 0, -1.0], rng.uniform(-1, 1)),
        "plane": mi.quadric_plane(rng.normal(size=3), rng.uniform(-1, 1)),
    }


def test_quadric_distance_roots_and_first_crossing():
    """P35: the returned distance is a root of f along the ray (residual at rounding level), f keeps the
    particle's sign before it (dense sampling: no earlier sign change), and +inf means no sign change at all."""
    rng = np.random.default_rng(35)
    n_hit = n_miss = 0
    for trial in range(300):
        for name, q in random_quadrics(rng).items():
            r = rng.uniform(-3, 3, 3)
            u = rng.normal(size=3); u /= np.linalg.norm(u)
            f0 = feval(q, r)
            if abs(f0) < 1e-6:
                continue
            sense = 1.0 if f0 > 0 else -1.0
            d = qdist(q, sense, r, u)
            s = np.linspace(0.0, 40.0 if d == INF else d, 4001)[1:-1]
            pts = r[None, :] + s[:, None] * u[None, :]
            fs = np.array([feval(q, p) for p in pts])
            assert np.all(fs * sense > -1e-9), (name, trial, d)
            if d == INF:
                n_miss += 1
                continue
            n_hit += 1
            scale = max(1.0, float(np.abs(q).max())) * max(1.0, d * d + float(r @ r))
            assert abs(feval(q, r + d * u)) <= 1e-11 * scale, (name, d, feval(q, r + d * u))
            assert feval(q, r + (d + 1e-6 * max(1.0, d)) * u) * sense < 0.0, name     # the sign does change there
    assert n_hit > 500 and n_miss > 300
    # on the surface: the logical side decides (c = 0): leaving -> +inf or the far root, entering -> the far root
    q = mi.quadric_sphere((0, 0, 0), 1.0)
    assert qdist(q, +1, (1, 0, 0), (1, 0, 0)) == INF                      # outside, moving away
    assert qdist(q, -1, (1, 0, 0), (-1, 0, 0)) == pytest.approx(2.0, abs=1e-15)   # inside, just entered: far side
    assert qdist(q, -1, (1, 0, 0), (1, 0, 0)) == 0.0                      # logically inside, moving out: crosses at once
    assert qdist(q, +1, (1, 0, 0), (-1, 0, 0)) == 0.0                     # logically outside, moving in
    assert qdist(q, +1, (1.0000000001, 0, 0), (0, 1, 0)) == INF           # tangent-like miss
    p = mi.quadric_plane((0, 0, 1), 2.0)
    assert qdist(p, -1, (0, 0, 0), (0, 0, 1)) == 2.0 and qdist(p, -1, (0, 0, 0), (0, 0, -1)) == INF
    assert qdist(p, -1, (0, 0, 0), (1, 0, 0)) == INF


@pytest.mark.parametrize("r", [0.5, 1.0, 2.0])
def test_sphere_escape_probability(r):
    """P36: uniform isotropic source in a purely absorbing sphere (Sigma_t = 1) in a void: the escape
    probability is 3/(8 r^3) (2 r^2 - 1 + (1 + 2r) e^{-2r}).  Pins the sphere distance, the logical region
    flip at the surface, the region materials and the ball source (source kind 3)."""
    N = 200_000
    c = (0.3, -0.2, 0.1)
    mats = mi._materials_1g([1.0, 1e-9], [0.0, 0.0], [1.0, 1e-9], [0, 0], [0, 0])
    cfg = mi.csg_problem(mats, [mi.quadric_sphere(c, r)], [([-1], 0), ([1], 1)], box=((-5, 5),) * 3,
                         source=mi.ball_source(c, r), n_hist=N, seed=36)
    o = Oracle(cfg).run()
    k = o.counters()
    P = 3 / (8 * r ** 3) * (2 * r * r - 1 + (1 + 2 * r) * math.exp(-2 * r))
    assert k["lost"] == 0 and k["leaks"] + k["captures"] == N
    assert abs(k["leaks"] / N - P) < 4 * math.sqrt(P * (1 - P) / N) + 1e-7
    assert k["crossings"] == k["leaks"] - 0 or abs(k["crossings"] - k["leaks"]) <= 2     # one sphere crossing per escape
    # with the materials exchanged nothing is absorbed in the ball
    cfg2 = mi.csg_problem(mats, [mi.quadric_sphere(c, r)], [([-1], 1), ([1], 0)], box=((-5, 5),) * 3,
                          source=mi.ball_source(c, r), n_hist=5_000, seed=36)
    k2 = Oracle(cfg2).run().counters()
    assert k2["captures"] + k2["leaks"] == 5_000 and k2["crossings"] == 5_000


def _ki2(x, n=4000):
    th = (np.arange(n) + 0.5) / n * (math.pi / 2)
    return float(np.sum(np.sin(th) * np.exp(-x / np.sin(th))) * (math.pi / 2 / n))


@pytest.mark.parametrize("axis", [(0, 0, 1), (1, 0, 0), (1, 2, 3), (-2, 1, 0.5)])
def test_cylinder_escape_from_its_axis_any_orientation(axis):
    """P37: isotropic point source on the axis of an infinite purely absorbing cylinder (Sigma_t R = 1.3):
    the escape probability is the Bickley function Ki2(Sigma_t R), whatever the orientation of the axis
    (cross terms D, E, F of the quadric) and wherever the axis passes."""
    N = 200_000
    R, sig = 0.65, 2.0
    p0 = np.array([0.4, -0.3, 0.2])
    a = np.array(axis, float) / np.linalg.norm(axis)
    mats = mi._materials_1g([sig, 1e-9], [0.0, 0.0], [sig, 1e-9], [0, 0], [0, 0])
    src = mi._point_source(tuple(p0 + 0.7 * a))
    cfg = mi.csg_problem(mats, [mi.quadric_cylinder(p0, a, R)], [([-1], 0), ([1], 1)], box=((-50, 50),) * 3,
                         source=src, n_hist=N, seed=37)
    k = Oracle(cfg).run().counters()
    P = _ki2(sig * R)
    assert k["lost"] == 0
    # (particles that escape the cylinder reach the box through 50 cm of near-void; a few fly along the axis
    # for more than the box: they are absorbed or leave through the end faces, both count below)
    esc = k["crossings"]
    assert abs(esc / N - P) < 4 * math.sqrt(P * (1 - P) / N) + 2e-3, (esc / N, P)


def test_lattice_cylinder_agrees_with_the_same_closed_form():
    """P37b: the lattice's z-cylinder (C.6, App. C.1) against the same Ki2: both geometry paths, one number."""
    N = 200_000
    R, sig = 0.54, 2.0
    mats = mi._materials_1g([sig, 1e-9], [0.0, 0.0], [sig, 1e-9], [0, 0], [0, 0])
    geom = dict(xs=np.array([0.0, 1.26]), ys=np.array([0.0, 1.26]), zs=np.array([-INF, INF]),
                mat_outer=np.full((1, 1, 1), 1, np.int32), mat_inner=np.full((1, 1, 1), 0, np.int32),
                radius=np.full((1, 1, 1), R), bc=np.zeros(6, np.int32))
    cfg = dict(name="pin_axis", materials=mats, geometry=geom, source=mi._point_source((0.63, 0.63, 0.0)),
               tally=dict(txs=geom["xs"].copy(), tys=geom["ys"].copy(), tzs=geom["zs"].copy(), tts=np.array([0.0, INF])),
               census=dict(t_census=np.zeros(0), comb_target=0), run=dict(seed=38, n_hist_per_batch=N, n_batch=1))
    k = Oracle(cfg).run().counters()
    P = _ki2(sig * R)
    assert abs(k["leaks"] / N - P) < 4 * math.sqrt(P * (1 - P) / N) + 1e-6


def test_slab_of_config2_rebuilt_from_quadric_planes():
    """P38: the four-region slab of config 2 as a CSG (three quadric planes inside the box [0, 20]) gives the
    region fluxes and leakage of the lattice version within 4 sigma (independent seeds), exactly one region
    change per interface crossing, and no lost particle."""
    N = 100_000
    lat = Oracle(mi.config2(n_hist=N, seed=1)).run()
    ref = mi.config2(n_hist=N, seed=2)
    planes = [mi.quadric_plane((1, 0, 0), x) for x in (5.0, 10.0, 15.0)]
    regions = [([-1], 0), ([1, -2], 1), ([2, -3], 2), ([3], 3)]
    cfg = mi.csg_problem(ref["materials"], planes, regions, box=((0.0, 20.0), (-INF, INF), (-INF, INF)),
                         source=ref["source"], tally=ref["tally"], t_census=ref["census"]["t_census"], n_hist=N, seed=2)
    csg = Oracle(cfg).run()
    a, b = lat.counters(), csg.counters()
    assert b["lost"] == 0
    for key in ("leaks", "captures", "collisions", "crossings", "census"):
        sig = math.sqrt(max(a[key], 1)) * 1.5          # (correlated within histories: generous)
        # the pulse sits ON the second plane: the coordinate lookup of the CSG puts every source particle on its
        # negative side, and the half that moves to +x crosses it at once (a flight of length 0); the lattice
        # looks its cell up with the direction (C.4)
        shift = N / 2 if key == "crossings" else 0.0
        extra = math.sqrt(N / 4) if key == "crossings" else 0.0
        assert abs(b[key] - a[key] - shift) < 4 * (math.sqrt(2) * sig + extra) + 5, (key, a[key], b[key])
    fa = lat.tally(0)[:, 0, 0, 0, :].sum(axis=0).reshape(4, 50).sum(axis=1)
    fb = csg.tally(0)[:, 0, 0, 0, :].sum(axis=0).reshape(4, 50).sum(axis=1)
    assert np.all(np.abs(fa - fb) < 0.03 * np.maximum(fa, fb) + 1e-3), (fa, fb)


@pytest.mark.parametrize("case", ["chasing", "two_intervals", "receding_exit"])
def test_attenuation_behind_a_moving_interface(case):
    """P39 (C.19): a beam (speed v = 2, direction +x, from x = 0 at t = 0) and a plane interface that moves
    along x.  chasing / two_intervals: void on the left of the interface X(t), absorber (Sigma = 0.7) on the
    right; the beam enters the absorber when 2 t = X(t) and the census at T finds exp(-Sigma v (T - t*)) of it.
    receding_exit: the absorber is on the LEFT of the interface; the beam is born in it and leaves it at t*:
    the fraction exp(-Sigma v t*) reaches the census.  A static interface would give other numbers."""
    N, v, sig, T = 100_000, 2.0, 0.7, 6.0
    mats = mi._materials_1g([sig, 1e-9], [0.0, 0.0], [sig, 1e-9], [0, 0], [0, 0], speed=v)
    if case == "chasing":
        tau = [0.0, 10.0]; X0 = 3.0; disp = [[[0, 0, 0], [10.0, 0, 0]]]            # V = 1 < v
        t_star = X0 / (v - 1.0); expect = math.exp(-sig * v * (T - t_star)); left, right = 1, 0
    elif case == "two_intervals":
        tau = [0.0, 1.0, 11.0]; X0 = 3.0; disp = [[[0, 0, 0], [1.5, 0, 0], [1.5 + 5.0, 0, 0]]]   # V = 1.5, then 0.5
        # interval 1: 2 t = 3 + 1.5 t -> t = 6 > 1: no; interval 2: 2 t = 4.5 + 0.5 (t - 1) -> t = 8/3
        t_star = 8.0 / 3.0; expect = math.exp(-sig * v * (T - t_star)); left, right = 1, 0
    else:
        tau = [0.0, 10.0]; X0 = 1.0; disp = [[[0, 0, 0], [5.0, 0, 0]]]             # V = 0.5
        t_star = X0 / (v - 0.5); expect = math.exp(-sig * v * t_star); left, right = 0, 1
    src = mi._point_source((0.0, 0.0, 0.0)); src["isotropic"] = 0
    cfg = mi.csg_problem(mats, [mi.quadric_plane((1, 0, 0), X0)], [([-1], left), ([1], right)],
                         box=((-INF, INF),) * 3, source=src, tally=None, t_census=[T], n_hist=N, seed=39,
                         motion=(tau, disp))
    cfg["tally"]["tts"] = np.array([0.0, T])
    o = Oracle(cfg).run()
    k = o.counters()
    assert k["lost"] == 0 and k["census"] + k["captures"] == N
    assert abs(k["census"] / N - expect) < 4 * math.sqrt(expect * (1 - expect) / N) + 1e-6, (k["census"] / N, expect)
    static = math.exp(-sig * v * (T - X0 / v)) if case != "receding_exit" else math.exp(-sig * X0)
    assert abs(static - expect) > 20 * math.sqrt(expect * (1 - expect) / N)
    # every history that lives through a break time stops there once; every survivor crosses the interface once
    if case == "two_intervals":
        assert k["crossings"] >= k["census"] * 2


def test_csg_rejects_bad_input():
    cfg = mi.csg_problem(mi._materials_1g([1.0], [0.5], [0.5], [0], [0]), [mi.quadric_sphere((0, 0, 0), 1.0)],
                         [([-1], 0), ([1], 0)], n_hist=10)
    Oracle(cfg).run()
    bad = dict(cfg); bad["csg"] = dict(cfg["csg"]); bad["csg"]["region_mat"] = np.array([0, 3], np.int32)
    with pytest.raises(ValueError):
        Oracle(bad)
    bad = dict(cfg); bad["csg"] = dict(cfg["csg"]); bad["csg"]["region_surf"] = cfg["csg"]["region_surf"].copy()
    bad["csg"]["region_surf"][0, 0] = 5
    with pytest.raises(ValueError):
        Oracle(bad)
    lat = mi.config2(n_hist=10); lat["csg"] = cfg["csg"]           # a lattice of four cells cannot hold a CSG
    with pytest.raises(ValueError):
        Oracle(lat)
    mv = dict(cfg); mv["motion"] = dict(tau=np.array([1.0, 0.5]), disp=np.zeros((1, 2, 3)))
    with pytest.raises(ValueError):
        Oracle(mv)
    # a geometry with a hole: the particle that enters it is lost and the run says so
    hole = mi.csg_problem(mi._materials_1g([1e-9], [0.0], [1e-9], [0], [0]), [mi.quadric_sphere((0, 0, 0), 1.0)],
                          [([-1], 0)], box=((-5, 5),) * 3, n_hist=10)
    o = Oracle(hole)
    with pytest.raises(RuntimeError):
        o.run()
    assert o.counters()["lost"] == 10
