"""Seeded synthetic input generators shared by the oracle and the CUDA path.

This module holds NONE of the method's arithmetic: it only builds the arrays
(materials, lattice geometry, source, tally mesh, census times, run sizes) that
both sides receive unchanged.  The five workloads are BASELINE.json configs
1..5 (lines 7-11) with the readings of DESIGN.md §3 (S11-S24, App. E); they
stand in for the paper's AZURV1 / slab / C5G7-pin / 3-D core problems
(PAPER.md:67, :91, :103), whose data are not available.
"""
from __future__ import annotations

import json
import os

import numpy as np

INF = float("inf")
XS_SEED = 20230507
_HERE = os.path.dirname(os.path.abspath(__file__))


def _one_cell_geometry(n_mat_outer=0):
    return dict(
        xs=np.array([-INF, INF]), ys=np.array([-INF, INF]), zs=np.array([-INF, INF]),
        mat_outer=np.full((1, 1, 1), n_mat_outer, np.int32),
        mat_inner=np.full((1, 1, 1), -1, np.int32),
        radius=np.zeros((1, 1, 1)), bc=np.zeros(6, np.int32),
    )


def _materials_1g(sigma_t, sigma_s, sigma_c, sigma_f, nu, speed=1.0):
    sigma_t = np.atleast_1d(np.asarray(sigma_t, float))
    M = sigma_t.size
    f = lambda a: np.atleast_1d(np.asarray(a, float)).reshape(M, 1)
    sf = f(sigma_f)
    return dict(
        sigma_t=sigma_t.reshape(M, 1), sigma_c=f(sigma_c), sigma_f=sf, nu=f(nu),
        sigma_s=np.atleast_1d(np.asarray(sigma_s, float)).reshape(M, 1, 1),
        chi=np.ones((M, 1)), speed=np.array([float(speed)]),
    )


def _point_source(pos=(0.0, 0.0, 0.0), G=1):
    pdf = np.zeros(G); pdf[0] = 1.0
    return dict(kind=0, lo=np.array(pos, float), hi=np.array(pos, float), isotropic=1,
                dir=np.array([1.0, 0.0, 0.0]), group_pdf=pdf, t0=0.0)


def infinite_medium(sigma_t=1.0, sigma_s=0.5, sigma_c=0.5, sigma_f=0.0, nu=0.0, speed=1.0,
                    t_edges=None, t_census=None, comb_target=0,
                    n_hist=100_000, n_batch=1, seed=0):
    """One infinite homogeneous 1-group cell; generic builder for configs 1, 3
    and the closed-form pins (P3, P5, P6)."""
    t_edges = np.array([0.0, INF]) if t_edges is None else np.asarray(t_edges, float)
    t_census = np.zeros(0) if t_census is None else np.asarray(t_census, float)
    return dict(
        name="infinite_medium",
        materials=_materials_1g(sigma_t, sigma_s, sigma_c, sigma_f, nu, speed),
        geometry=_one_cell_geometry(),
        source=_point_source(),
        tally=dict(txs=np.array([-INF, INF]), tys=np.array([-INF, INF]),
                   tzs=np.array([-INF, INF]), tts=t_edges),
        census=dict(t_census=t_census, comb_target=int(comb_target)),
        run=dict(seed=int(seed), n_hist_per_batch=int(n_hist), n_batch=int(n_batch)),
    )


def config1(n_hist=100_000, n_batch=1, seed=0):
    """BASELINE.json:7 — infinite medium, Sigma_t 1, Sigma_s 0.5, Sigma_a 0.5."""
    c = infinite_medium(n_hist=n_hist, n_batch=n_batch, seed=seed)
    c["name"] = "config1"
    return c


def slab(sigma_t, sigma_s, edges, src_x, beam=False, tally_x=None, tally_t=None,
         t_end=None, n_hist=100_000, n_batch=1, seed=0):
    """1-D slab along x with vacuum faces; y,z infinite."""
    sigma_t = np.asarray(sigma_t, float); sigma_s = np.asarray(sigma_s, float)
    edges = np.asarray(edges, float)
    nreg = sigma_t.size
    geom = dict(
        xs=edges, ys=np.array([-INF, INF]), zs=np.array([-INF, INF]),
        mat_outer=np.arange(nreg, dtype=np.int32).reshape(1, 1, nreg),
        mat_inner=np.full((1, 1, nreg), -1, np.int32),
        radius=np.zeros((1, 1, nreg)), bc=np.zeros(6, np.int32),
    )
    src = _point_source((src_x, 0.0, 0.0))
    if beam:
        src["isotropic"] = 0
    tally_x = edges[[0, -1]] if tally_x is None else np.asarray(tally_x, float)
    if tally_t is None:
        tally_t = np.array([0.0, INF if t_end is None else t_end])
    t_census = np.zeros(0) if t_end is None else np.array([float(t_end)])
    return dict(
        name="slab",
        materials=_materials_1g(sigma_t, sigma_s, sigma_t - sigma_s, np.zeros(nreg), np.zeros(nreg)),
        geometry=geom, source=src,
        tally=dict(txs=tally_x, tys=np.array([-INF, INF]), tzs=np.array([-INF, INF]),
                   tts=np.asarray(tally_t, float)),
        census=dict(t_census=t_census, comb_target=0),
        run=dict(seed=int(seed), n_hist_per_batch=int(n_hist), n_batch=int(n_batch)),
    )


def config2(n_hist=1_000_000, n_batch=1, seed=0, nx_tally=200, nt_tally=100):
    """BASELINE.json:8 — 4-region slab, pulse at the x=10 interface (S7, S12)."""
    tx = np.array([j * 0.1 for j in range(201)])
    if nx_tally != 200:
        assert 200 % nx_tally == 0
        tx = tx[:: 200 // nx_tally]
    tt = np.array([j * 0.2 for j in range(101)])
    if nt_tally != 100:
        assert 100 % nt_tally == 0
        tt = tt[:: 100 // nt_tally]
    full = np.array([j * 0.1 for j in range(201)])
    edges = full[[0, 50, 100, 150, 200]]       # geometry planes := tally table values
    st = np.array([1.0, 0.5, 2.0, 1.0])
    ss = np.array([0.9, 0.5, 0.2, 0.99]) * st
    c = slab(st, ss, edges, src_x=edges[2], tally_x=tx, tally_t=tt, t_end=tt[-1],
             n_hist=n_hist, n_batch=n_batch, seed=seed)
    c["name"] = "config2"
    return c


def config3(n_hist=1_000_000, n_batch=1, seed=0, comb_target=None):
    """BASELINE.json:9 — supercritical infinite medium, 20 census steps + comb (S13)."""
    tk = np.array([0.1 * k for k in range(21)])
    c = infinite_medium(1.0, 0.4, 0.3, 0.3, 2.5, 1.0, t_edges=tk, t_census=tk[1:],
                        comb_target=n_hist if comb_target is None else comb_target,
                        n_hist=n_hist, n_batch=n_batch, seed=seed)
    c["name"] = "config3"
    return c


def seeded_materials(n_mat, fissile, G=7, nusf_scale=1.0, rng=None):
    """App. E recipe (S11, S19, S20, S24): seeded random 7-group materials."""
    rng = np.random.default_rng(XS_SEED) if rng is None else rng
    st = np.zeros((n_mat, G)); ss = np.zeros((n_mat, G, G)); sf = np.zeros((n_mat, G))
    sc = np.zeros((n_mat, G)); nu = np.zeros((n_mat, G)); chi = np.zeros((n_mat, G))
    for m in range(n_mat):
        st[m] = rng.uniform(0.2, 2.0, G)
        c = rng.uniform(0.3, 0.95, G)
        W = np.triu(rng.uniform(0.0, 1.0, (G, G)))           # g' >= g only (downscatter)
        ss[m] = (c * st[m])[:, None] * W / W.sum(axis=1, keepdims=True)
        srow = np.zeros(G)
        for g in range(G):                                     # ascending sequential sum
            acc = 0.0
            for j in range(G):
                acc = acc + ss[m, g, j]
            srow[g] = acc
        sa = st[m] - srow
        if m in fissile:
            nusf = rng.uniform(0.0, 0.5, G) * nusf_scale
            nu[m] = 2.5
            sf[m] = np.minimum(nusf / 2.5, sa)
            x = rng.uniform(0.0, 1.0, 3)
            chi[m, :3] = x / x.sum()
            chi[m, 2] = 1.0 - (chi[m, 0] + chi[m, 1])
        sc[m] = sa - sf[m]
    speed = np.array([2e9 * 10.0 ** (-4.0 * g / 6.0) for g in range(G)])
    return dict(sigma_t=st, sigma_c=sc, sigma_f=sf, nu=nu, sigma_s=ss, chi=chi, speed=speed), rng


def config4(n_hist=1_000_000, n_batch=10, seed=0, t_end=5e-5):
    """BASELINE.json:10 — 17x17 pin lattice, 7 groups, reflective box (S15, S16, S23)."""
    mats, _ = seeded_materials(2, fissile=(0,))
    tab = np.array([j * 0.42 for j in range(52)])
    planes = tab[::3]
    n = 17
    zs = np.array([0.0, 21.42])
    geom = dict(
        xs=planes, ys=planes.copy(), zs=zs,
        mat_outer=np.full((1, n, n), 1, np.int32), mat_inner=np.zeros((1, n, n), np.int32),
        radius=np.full((1, n, n), 0.54), bc=np.ones(6, np.int32),
    )
    src = dict(kind=2, lo=np.array([planes[0], planes[0], zs[0]]),
               hi=np.array([planes[-1], planes[-1], zs[1]]), isotropic=1,
               dir=np.array([1.0, 0.0, 0.0]), group_pdf=mats["chi"][0].copy(), t0=0.0)
    tt = np.array([t_end * j / 10 for j in range(11)])
    return dict(
        name="config4", materials=mats, geometry=geom, source=src,
        tally=dict(txs=tab, tys=tab.copy(), tzs=zs.copy(), tts=tt),
        census=dict(t_census=tt[-1:].copy(), comb_target=0),
        run=dict(seed=int(seed), n_hist_per_batch=int(n_hist), n_batch=int(n_batch)),
    )


def config5_scale():
    """nu*Sigma_f multiplier of S17, written by mcdc_inputs/calibrate_config5.py."""
    with open(os.path.join(_HERE, "config5_scale.json")) as f:
        return float(json.load(f)["nusf_scale"])


def config5(n_hist=10_000_000, n_batch=10, seed=0, n_vox=64, nusf_scale=None,
            comb_target=None, n_steps=20, dt=5e-6):
    """BASELINE.json:11 — 64^3 voxel box, 8 random 7-group materials, 20 census + comb (S17, S18)."""
    if nusf_scale is None:
        nusf_scale = config5_scale()
    mats, rng = seeded_materials(8, fissile=(0, 1, 2), nusf_scale=nusf_scale)
    vox = rng.integers(0, 8, (64, 64, 64), dtype=np.int8).astype(np.int32)
    vox = np.ascontiguousarray(vox[:n_vox, :n_vox, :n_vox])
    planes = np.array([float(i) for i in range(n_vox + 1)])
    geom = dict(
        xs=planes, ys=planes.copy(), zs=planes.copy(), mat_outer=vox,
        mat_inner=np.full(vox.shape, -1, np.int32), radius=np.zeros(vox.shape),
        bc=np.zeros(6, np.int32),
    )
    pdf = np.zeros(7); pdf[0] = 1.0
    src = dict(kind=1, lo=np.zeros(3), hi=np.full(3, float(n_vox)), isotropic=1,
               dir=np.array([1.0, 0.0, 0.0]), group_pdf=pdf, t0=0.0)
    tt = np.array([dt * k for k in range(n_steps + 1)])
    return dict(
        name="config5", materials=mats, geometry=geom, source=src,
        tally=dict(txs=planes.copy(), tys=planes.copy(), tzs=planes.copy(), tts=tt),
        census=dict(t_census=tt[1:].copy(),
                    comb_target=int(n_hist if comb_target is None else comb_target)),
        run=dict(seed=int(seed), n_hist_per_batch=int(n_hist), n_batch=int(n_batch)),
    )


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def config(k, **kw):
    return CONFIGS[int(k)](**kw)


def infinite_multigroup(mats, m, group_pdf, n_hist=100_000, n_batch=1, seed=0):
    """Infinite homogeneous medium made of material m of a multigroup set (pin P10)."""
    G = mats["sigma_t"].shape[1]
    one = {k: np.ascontiguousarray(mats[k][m:m + 1]) for k in
           ("sigma_t", "sigma_c", "sigma_f", "nu", "sigma_s", "chi")}
    one["speed"] = mats["speed"].copy()
    src = _point_source(G=G)
    src["group_pdf"] = np.asarray(group_pdf, float)
    return dict(
        name="infinite_multigroup", materials=one, geometry=_one_cell_geometry(), source=src,
        tally=dict(txs=np.array([-INF, INF]), tys=np.array([-INF, INF]),
                   tzs=np.array([-INF, INF]), tts=np.array([0.0, INF])),
        census=dict(t_census=np.zeros(0), comb_target=0),
        run=dict(seed=int(seed), n_hist_per_batch=int(n_hist), n_batch=int(n_batch)),
    )


def delayed(cfg, nu_delayed, decay, chi_delayed=None):
    """Adds delayed-neutron data (DESIGN.md §3 C.16): nu_delayed [M][G][J] (part of
    the TOTAL nu already in the materials), decay [M][J], chi_delayed [M][J][G] (default: the prompt
    spectrum of the material)."""
    cfg = dict(cfg)
    m = cfg["materials"]
    M, G = np.asarray(m["sigma_t"]).shape
    nud = np.asarray(nu_delayed, float).reshape(M, G, -1)
    J = nud.shape[-1]
    lam = np.asarray(decay, float).reshape(M, J)
    chd = (np.repeat(np.asarray(m["chi"], float)[:, None, :], J, axis=1) if chi_delayed is None
           else np.asarray(chi_delayed, float).reshape(M, J, G))
    cfg["delayed"] = dict(nu_delayed=nud.copy(), decay=lam.copy(), chi_delayed=chd.copy())
    cfg["name"] = cfg["name"] + "_dn"
    return cfg


def seeded_delayed(cfg, J=6, beta=0.0065, seed=20230508, lambda_range=(0.0125, 3.0), time_scale=1.0):
    """Seeded stand-in for a six-group delayed-neutron set (the C5G7-TD data are not available): delayed
    fraction beta of nu split over J groups with random shares, decay constants log-spaced over
    lambda_range (1/s, the usual span) divided by time_scale, delayed spectra softer than the prompt one
    (random over the first four groups)."""
    rng = np.random.default_rng(seed)
    m = cfg["materials"]
    M, G = np.asarray(m["sigma_t"]).shape
    share = rng.random(J) + 0.2
    share = share / share.sum()
    nud = beta * np.asarray(m["nu"], float)[:, :, None] * share[None, None, :]
    lam = np.tile(np.geomspace(lambda_range[0], lambda_range[1], J) / time_scale, (M, 1))
    chd = np.zeros((M, J, G))
    hi = min(G, 4)
    for mm in range(M):
        for j in range(J):
            w = rng.random(hi) + 0.1
            chd[mm, j, :hi] = w / w.sum()
            chd[mm, j, hi - 1] += 1.0 - chd[mm, j].sum()
    return delayed(cfg, nud, lam, chd)


def implicit_capture(cfg, w_roulette=0.0, w_survive=1.0):
    """Switches implicit capture on (DESIGN.md §3 C.15): weight roulette below w_roulette
    (0 = off) back to w_survive; the census comb becomes the weighted comb."""
    cfg = dict(cfg)
    cfg["implicit_capture"] = dict(w_roulette=float(w_roulette), w_survive=float(w_survive))
    cfg["name"] = cfg["name"] + "_ic"
    return cfg


def eigenvalue(cfg, n_inactive, n_active, k0=1.0):
    """Turns a time-independent fixed-source config into a k-eigenvalue run (
    DESIGN.md §3 C.14): n_inactive + n_active fission generations of n_hist_per_batch particles,
    the first generation drawn from the config's source."""
    assert len(cfg["census"]["t_census"]) == 0, "eigenvalue mode is time-independent"
    cfg = dict(cfg)
    cfg["eigenvalue"] = dict(n_inactive=int(n_inactive), n_active=int(n_active), k0=float(k0))
    cfg["name"] = cfg["name"] + "_keig"
    return cfg


def fissile_slab(sigma_t=1.0, sigma_s=0.5, sigma_f=0.2, nu=2.5, width=6.0, nx_tally=12,
                 n_hist=20_000, n_batch=1, seed=0):
    """Bare 1-group fissile slab with vacuum faces (an eigenvalue pin with leakage); uniform first
    generation."""
    c = slab([sigma_t], [sigma_s], [0.0, float(width)], src_x=0.0,
             tally_x=[width * j / nx_tally for j in range(nx_tally + 1)],
             n_hist=n_hist, n_batch=n_batch, seed=seed)
    c["materials"] = _materials_1g(sigma_t, sigma_s, sigma_t - sigma_s - sigma_f, sigma_f, nu)
    c["source"].update(kind=1, lo=np.array([0.0, 0.0, 0.0]), hi=np.array([float(width), 0.0, 0.0]))
    c["name"] = "fissile_slab"
    return c


def pin_cell_eigenvalue(n_hist=100_000, n_inactive=50, n_active=100, k0=1.0, n_batch=1, seed=0,
                        mesh=(20, 20, 100), nusf_scale=7.0):
    """Stand-in for the paper's k-eigenvalue benchmark ("multigroup infinite pin cell
    criticality problem ... 50 inactive and 100 active cycles with 10^5 particles per cycle", flux on a
    20 x 20 x 100 x 7 mesh): one reflective pin cell (radius 0.54, pitch 1.26, height 21.42) of the
    config-4 materials (the C5G7 data are not available) with the fuel's nu*Sigma_f draw times 7, which
    puts k near 1 (found with the oracle: 0.19 at 1, 0.94 at 6, 1.11 at 10); first generation uniform
    in the fuel."""
    mats, _ = seeded_materials(2, fissile=(0,), nusf_scale=nusf_scale)
    nx, ny, nz = mesh
    tx = np.array([j * (1.26 / nx) for j in range(nx + 1)])
    ty = np.array([j * (1.26 / ny) for j in range(ny + 1)])
    tz = np.array([j * (21.42 / nz) for j in range(nz + 1)])
    geom = dict(
        xs=tx[[0, -1]].copy(), ys=ty[[0, -1]].copy(), zs=tz[[0, -1]].copy(),
        mat_outer=np.full((1, 1, 1), 1, np.int32), mat_inner=np.zeros((1, 1, 1), np.int32),
        radius=np.full((1, 1, 1), 0.54), bc=np.ones(6, np.int32),
    )
    src = dict(kind=2, lo=np.array([tx[0], ty[0], tz[0]]), hi=np.array([tx[-1], ty[-1], tz[-1]]),
               isotropic=1, dir=np.array([1.0, 0.0, 0.0]), group_pdf=mats["chi"][0].copy(), t0=0.0)
    cfg = dict(
        name="pin_cell", materials=mats, geometry=geom, source=src,
        tally=dict(txs=tx, tys=ty, tzs=tz, tts=np.array([0.0, INF])),
        census=dict(t_census=np.zeros(0), comb_target=0),
        run=dict(seed=int(seed), n_hist_per_batch=int(n_hist), n_batch=int(n_batch)),
    )
    return eigenvalue(cfg, n_inactive, n_active, k0)


def dogleg_duct(n_hist=100_000, n_batch=1, seed=0, n_cell=(6, 10, 6), pitch=10.0, t_source=50.0, t_end=200.0,
                nt=20, n_census=4, sub=2):
    """Synthetic stand-in for the paper's time-dependent dog-leg void duct problem: the
    paper fixes only the speed (1 cm/s), the source window (first 50 s), the end time (200 s), the
    track-length mesh tally, 1e8 histories and implicit capture; the benchmark's geometry and cross
    sections (its ref [14]) are not available, so this is OUR OWN box: n_cell cubic cells of `pitch` cm,
    a source cell in the corner at the origin, a void duct that leaves it along +y, turns along +x,
    then +z, then +y again to the far face, shield everywhere else; reflective faces at x = y = z = 0,
    vacuum outside; materials: source and shield Sigma_t = 0.1 with 50 % scattering, void Sigma_t = 1e-4
    with 50 % scattering.  Tally: `sub` bins per cell per axis x nt time bins; n_census census steps
    (no comb: the population only falls)."""
    nx, ny, nz = n_cell
    mat = np.full((nz, ny, nx), 1, np.int32)             # 1 = shield
    duct = [(0, j, 0) for j in range(1, ny // 2)]
    duct += [(i, ny // 2 - 1, 0) for i in range(0, nx // 2)]
    duct += [(nx // 2 - 1, ny // 2 - 1, k) for k in range(0, nz // 2)]
    duct += [(nx // 2 - 1, j, nz // 2 - 1) for j in range(ny // 2 - 1, ny)]
    for (i, j, k) in duct:
        mat[k, j, i] = 2                                 # 2 = void
    mat[0, 0, 0] = 0                                     # 0 = source cell
    st = np.array([[0.1], [0.1], [1e-4]])
    mats = dict(sigma_t=st, sigma_c=0.5 * st, sigma_f=np.zeros((3, 1)), nu=np.zeros((3, 1)),
                sigma_s=(0.5 * st)[:, :, None].copy(), chi=np.ones((3, 1)), speed=np.array([1.0]))
    xs, ys, zs = (np.array([pitch * i for i in range(n + 1)]) for n in (nx, ny, nz))
    geom = dict(xs=xs, ys=ys, zs=zs, mat_outer=mat, mat_inner=np.full((nz, ny, nx), -1, np.int32),
                radius=np.zeros((nz, ny, nx)), bc=np.array([1, 0, 1, 0, 1, 0], np.int32))
    src = dict(kind=1, lo=np.zeros(3), hi=np.full(3, pitch), isotropic=1, dir=np.array([1.0, 0.0, 0.0]),
               group_pdf=np.ones(1), t0=0.0, t_end=float(t_source))
    tx, ty, tz = (np.array([(pitch / sub) * i for i in range(n * sub + 1)]) for n in (nx, ny, nz))
    tts = np.array([t_end * j / nt for j in range(nt + 1)])
    assert nt % n_census == 0
    t_census = tts[nt // n_census::nt // n_census].copy()
    return dict(
        name="dogleg_duct", materials=mats, geometry=geom, source=src,
        tally=dict(txs=tx, tys=ty, tzs=tz, tts=tts),
        census=dict(t_census=t_census, comb_target=0),
        run=dict(seed=int(seed), n_hist_per_batch=int(n_hist), n_batch=int(n_batch)),
    )


# ---- quadric-surface CSG (DESIGN.md C.18) and moving surfaces (C.19): array builders only ----
def quadric_plane(n, d):
    """n . r - d (positive on the side n points to)."""
    q = np.zeros(10); q[6:9] = np.asarray(n, float); q[9] = -float(d)
    return q


def quadric_sphere(c, R):
    """|r - c|^2 - R^2."""
    c = np.asarray(c, float)
    q = np.zeros(10); q[0:3] = 1.0; q[6:9] = -2.0 * c; q[9] = float(c @ c - R * R)
    return q


def quadric_cylinder(p0, axis, R):
    """|r - p0|^2 - ((r - p0) . a)^2 - R^2 for a unit axis a through p0 (any orientation)."""
    p0 = np.asarray(p0, float); a = np.asarray(axis, float); a = a / np.linalg.norm(a)
    M = np.eye(3) - np.outer(a, a)
    q = np.zeros(10)
    q[0], q[1], q[2] = M[0, 0], M[1, 1], M[2, 2]
    q[3], q[4], q[5] = 2 * M[0, 1], 2 * M[1, 2], 2 * M[2, 0]
    g = -2.0 * M @ p0
    q[6:9] = g; q[9] = float(p0 @ M @ p0 - R * R)
    return q


def quadric_general(M, g, k):
    """r^T M r + g . r + k for a symmetric 3x3 M."""
    M = np.asarray(M, float)
    q = np.zeros(10)
    q[0], q[1], q[2] = M[0, 0], M[1, 1], M[2, 2]
    q[3], q[4], q[5] = 2 * M[0, 1], 2 * M[1, 2], 2 * M[2, 0]
    q[6:9] = np.asarray(g, float); q[9] = float(k)
    return q


def csg_problem(materials, surfaces, regions, box=((-INF, INF),) * 3, bc=(0,) * 6, source=None, tally=None,
                t_census=(), comb_target=0, n_hist=100_000, n_batch=1, seed=0, motion=None, name="csg"):
    """One lattice cell (the box) divided into regions by quadric surfaces.  regions: list of
    (signed surface list, material): +k / -k = positive / negative side of surface k (1-based)."""
    surfaces = np.asarray(surfaces, float).reshape(-1, 10)
    rs = np.zeros((len(regions), 8), np.int32)
    rm = np.zeros(len(regions), np.int32)
    for i, (lst, m) in enumerate(regions):
        rs[i, :len(lst)] = lst; rm[i] = m
    xs, ys, zs = (np.array(b, float) for b in box)
    geom = dict(xs=xs, ys=ys, zs=zs, mat_outer=np.zeros((1, 1, 1), np.int32), mat_inner=np.full((1, 1, 1), -1, np.int32),
                radius=np.zeros((1, 1, 1)), bc=np.asarray(bc, np.int32))
    G = np.asarray(materials["sigma_t"]).shape[1]
    if source is None:
        source = _point_source(G=G)
    if tally is None:
        tally = dict(txs=xs.copy(), tys=ys.copy(), tzs=zs.copy(), tts=np.array([0.0, INF]))
    cfg = dict(name=name, materials=materials, geometry=geom, source=source, tally=tally,
               census=dict(t_census=np.asarray(t_census, float), comb_target=int(comb_target)),
               run=dict(seed=int(seed), n_hist_per_batch=int(n_hist), n_batch=int(n_batch)),
               csg=dict(coef=surfaces, region_surf=rs, region_mat=rm))
    if motion is not None:
        cfg["motion"] = dict(tau=np.asarray(motion[0], float), disp=np.asarray(motion[1], float))
    return cfg


def ball_source(centre, radius, G=1, t0=0.0):
    """Source kind 3: uniform in a ball, isotropic."""
    pdf = np.zeros(G); pdf[0] = 1.0
    return dict(kind=3, lo=np.asarray(centre, float), hi=np.array([float(radius), 0.0, 0.0]), isotropic=1,
                dir=np.array([1.0, 0.0, 0.0]), group_pdf=pdf, t0=float(t0))
