"""Pins of the oracle's building blocks against things other than itself
(P1 Philox, P2 math functions, P12 DDA, P13 cylinder, P14 comb)."""
import ctypes as C
import math
import os
import subprocess
import sys

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
_dp = C.POINTER(C.c_double)
U32x = lambda *v: (C.c_uint32 * len(v))(*v)


def _philox(olib, key, ctr):
    out = (C.c_uint32 * 4)()
    olib.oracle_philox4x32_10(U32x(*key), U32x(*ctr), out)
    return tuple(out)


@pytest.fixture(scope="module")
def reflib(tmp_path_factory):
    """Library Philox implementations on the box: cuRAND header (host path) and torch's engine."""
    import torch
    tdir = os.path.join(os.path.dirname(torch.__file__), "include")
    so = str(tmp_path_factory.mktemp("philox") / "philox_ref.so")
    cmd = ["g++", "-O1", "-std=c++17", "-shared", "-fPIC", "-DWITH_TORCH",
           "-I/usr/local/cuda/include", "-I" + tdir, "-o", so,
           os.path.join(HERE, "helpers", "philox_ref.cpp")]
    subprocess.run(cmd, check=True)
    L = C.CDLL(so)
    L.ref_torch_philox.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(C.c_uint32)]
    return L


def test_philox_matches_curand_and_torch(olib, reflib):
    rng = np.random.default_rng(1)
    cases = [((0, 0), (0, 0, 0, 0)), ((0xFFFFFFFF,) * 2, (0xFFFFFFFF,) * 4)]
    for _ in range(10000):
        w = rng.integers(0, 2**32, 6, dtype=np.uint64)
        cases.append(((int(w[0]), int(w[1])), tuple(int(x) for x in w[2:])))
    for key, ctr in cases:
        mine = _philox(olib, key, ctr)
        out = (C.c_uint32 * 4)()
        reflib.ref_curand_philox(U32x(*key), U32x(*ctr), out)
        assert mine == tuple(out)
        seed = key[0] | (key[1] << 32)
        off = ctr[0] | (ctr[1] << 32)
        sub = ctr[2] | (ctr[3] << 32)
        reflib.ref_torch_philox(seed, sub, off, out)
        assert mine == tuple(out)


def test_philox_avalanche(olib):
    """Independent sanity property: flipping one counter bit flips about half the output bits."""
    rng = np.random.default_rng(2)
    flips = []
    for _ in range(500):
        w = [int(x) for x in rng.integers(0, 2**32, 6, dtype=np.uint64)]
        a = _philox(olib, w[:2], w[2:])
        w[2 + int(rng.integers(0, 4))] ^= 1 << int(rng.integers(0, 32))
        b = _philox(olib, w[:2], w[2:])
        flips.append(sum(bin(x ^ y).count("1") for x, y in zip(a, b)))
    assert abs(np.mean(flips) - 64.0) < 1.5


def test_uniform52_exact_and_open(olib):
    u = olib.oracle_uniform52
    assert u(0, 0) == 2.0**-53
    assert u(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0**-53
    assert u(0, 0xFFF) == 2.0**-53                 # low 12 bits are dropped
    assert u(0x80000000, 0) == 0.5 + 2.0**-53
    for hi, lo in [(1, 0), (0, 0x1000), (0xFFFFFFFF, 0xFFFFF000), (12345, 0xABCDE000)]:
        k = (hi << 20) | (lo >> 12)
        from fractions import Fraction
        assert Fraction(u(hi, lo)) == (Fraction(k) + Fraction(1, 2)) / 2**52   # exact in binary64
        assert u(hi, lo) + u(0xFFFFFFFF - hi, 0xFFFFFFFF - lo) == 1.0           # symmetric


def _ulp_err(got, ref):
    return abs(got - ref) / math.ulp(ref) if ref != 0 else abs(got) / 5e-324


def test_log_vs_libm(olib):
    rng = np.random.default_rng(3)
    xs = list(rng.uniform(0, 1, 200000)) + list(2.0 ** -rng.uniform(0, 53, 50000))
    xs += [2.0**-53, 1.0 - 2.0**-53, 0.5, 1.0, math.sqrt(0.5), 0.7071067811865476, 0.7071067811865475]
    worst = 0.0
    for x in xs:
        x = float(x)
        if x <= 0.0:
            continue
        got, ref = olib.oracle_log(x), math.log(x)
        if ref == 0.0:
            assert got == 0.0
            continue
        worst = max(worst, abs(got - ref) / max(math.ulp(ref), 2.0**-53 * 2**-52))
    assert worst <= 4.0, worst
    assert olib.oracle_log(1.0) == 0.0


def test_sincos2pi_vs_libm(olib):
    rng = np.random.default_rng(4)
    us = list(rng.uniform(0, 1, 200000)) + [2.0**-53, 1 - 2.0**-53, 0.125, 0.25, 0.375, 0.5, 0.625, 0.75, 0.875]
    c, s = C.c_double(), C.c_double()
    worst = 0.0
    for u in us:
        u = float(u)
        olib.oracle_sincos2pi(u, C.byref(c), C.byref(s))
        # reference angle reduced exactly first, so libm's argument error does not enter
        q4 = 4.0 * u
        k = int(q4); r = q4 - k
        rc, rs = math.cos(r * (math.pi / 2)), math.sin(r * (math.pi / 2))
        ref_c, ref_s = [(rc, rs), (-rs, rc), (-rc, -rs), (rs, -rc)][k & 3]
        # absolute error in units of 2^-53 (values are <= 1)
        worst = max(worst, abs(c.value - ref_c) / 2.0**-53, abs(s.value - ref_s) / 2.0**-53)
        assert abs(c.value * c.value + s.value * s.value - 1.0) <= 4 * 2.0**-52
    assert worst <= 4.0, worst
    olib.oracle_sincos2pi(0.25, C.byref(c), C.byref(s))
    assert (abs(c.value), s.value) == (0.0, 1.0)
    olib.oracle_sincos2pi(0.5, C.byref(c), C.byref(s))
    assert (c.value, abs(s.value)) == (-1.0, 0.0)


def test_cylinder_distance_bruteforce(olib):
    """P13: returned root satisfies the circle equation; cross-check against bisection."""
    rng = np.random.default_rng(5)
    R, cx, cy = 0.54, 0.63, 0.63
    for _ in range(5000):
        inside = int(rng.integers(0, 2))
        ang = rng.uniform(0, 2 * np.pi)
        rad = R * math.sqrt(rng.uniform(0, 1)) if inside else rng.uniform(R * 1.0001, 3 * R)
        x, y = cx + rad * math.cos(ang), cy + rad * math.sin(ang)
        mu = rng.uniform(-1, 1); ph = rng.uniform(0, 2 * np.pi)
        q = math.sqrt(1 - mu * mu)
        ux, uy = mu, q * math.cos(ph)               # projected direction, |.| <= 1
        d = olib.oracle_cyl_distance(x, y, ux, uy, cx, cy, R, inside)
        f = lambda s: (x + s * ux - cx) ** 2 + (y + s * uy - cy) ** 2 - R * R
        if math.isinf(d):
            assert not inside
            # brute force: the ray never gets inside
            ss = np.linspace(0, 10, 20001)
            assert np.all((x + ss * ux - cx) ** 2 + (y + ss * uy - cy) ** 2 >= R * R * (1 - 1e-9))
            continue
        assert d >= 0.0
        assert abs(f(d)) <= 1e-12 * max(1.0, d * d)
        # first crossing: no sign change of f before d
        ss = np.linspace(0, d, 400)[1:-1]
        vals = (x + ss * ux - cx) ** 2 + (y + ss * uy - cy) ** 2 - R * R
        assert np.all(vals < 1e-12) if inside else np.all(vals > -1e-12)


def _march(olib, mesh, pos, t, u, v, d, cap=4096):
    tx, ty, tz, tt = (np.ascontiguousarray(a, float) for a in mesh)
    bins = (C.c_int64 * cap)(); lens = (C.c_double * cap)()
    P = (C.c_double * 3)(*pos); U = (C.c_double * 3)(*u)
    n = olib.oracle_march(tx.ctypes.data_as(_dp), len(tx) - 1, ty.ctypes.data_as(_dp), len(ty) - 1,
                          tz.ctypes.data_as(_dp), len(tz) - 1, tt.ctypes.data_as(_dp), len(tt) - 1,
                          P, t, U, v, d, bins, lens, cap)
    return n, np.array(bins[:max(n, 0)]), np.array(lens[:max(n, 0)])


def test_march_vs_dense_sampling(olib):
    """P12: DDA segment lengths equal the bin occupancy of a densely sampled ray; sum = d."""
    rng = np.random.default_rng(6)
    for _ in range(300):
        nx, ny, nz, nt = (int(rng.integers(1, 7)) for _ in range(4))
        mk = lambda n, lo, hi: np.concatenate([[lo], np.sort(rng.uniform(lo, hi, n - 1)), [hi]])
        mesh = (mk(nx, 0, 4), mk(ny, 0, 3), mk(nz, 0, 5), mk(nt, 0, 2))
        pos = [rng.uniform(0.1, 3.9), rng.uniform(0.1, 2.9), rng.uniform(0.1, 4.9)]
        mu = rng.uniform(-1, 1); ph = rng.uniform(0, 2 * np.pi); q = math.sqrt(1 - mu * mu)
        u = [mu, q * math.cos(ph), q * math.sin(ph)]
        v = rng.uniform(0.5, 3.0); t = rng.uniform(0, 1.0)
        # longest flight staying inside the mesh in space and time
        dmax = min([((hi if ui > 0 else lo) - p) / ui for p, ui, lo, hi in
                    zip(pos, u, (0, 0, 0), (4, 3, 5)) if ui != 0] + [(2 - t) * v])
        d = dmax * rng.uniform(0.05, 0.999)
        n, bins, lens = _march(olib, mesh, pos, t, u, v, d)
        assert n >= 1 and np.all(lens > 0)
        assert abs(lens.sum() - d) <= 1e-12 * max(d, 1.0)
        K = 100000
        s = (np.arange(K) + 0.5) * (d / K)
        jx = np.searchsorted(mesh[0], pos[0] + s * u[0], side="right") - 1
        jy = np.searchsorted(mesh[1], pos[1] + s * u[1], side="right") - 1
        jz = np.searchsorted(mesh[2], pos[2] + s * u[2], side="right") - 1
        jt = np.searchsorted(mesh[3], t + s / v, side="right") - 1
        flat = ((jt * nz + jz) * ny + jy) * nx + jx
        ref = np.bincount(flat, minlength=nx * ny * nz * nt) * (d / K)
        got = np.zeros_like(ref); np.add.at(got, bins, lens)
        assert np.all(np.abs(got - ref) <= 2.5 * d / K * 4)


def test_march_on_plane_direction_aware(olib):
    """S7: a start exactly on a mesh plane goes to the lower bin when moving down, else upper."""
    mesh = (np.array([0.0, 1.0, 2.0]), np.array([-np.inf, np.inf]), np.array([-np.inf, np.inf]),
            np.array([0.0, np.inf]))
    n, b, l = _march(olib, mesh, [1.0, 0, 0], 0.0, [-1.0, 0, 0], 1.0, 0.5)
    assert (n, list(b), list(l)) == (1, [0], [0.5])
    n, b, l = _march(olib, mesh, [1.0, 0, 0], 0.0, [1.0, 0, 0], 1.0, 0.5)
    assert (n, list(b), list(l)) == (1, [1], [0.5])
    n, b, l = _march(olib, mesh, [1.0, 0, 0], 0.0, [0.0, 1.0, 0], 1.0, 0.5)
    assert (n, list(b), list(l)) == (1, [1], [0.5])
    # flight ending exactly on a plane does not create a zero-width crossing
    n, b, l = _march(olib, mesh, [0.25, 0, 0], 0.0, [1.0, 0, 0], 1.0, 0.75)
    assert (n, list(b), list(l)) == (1, [0], [0.75])
    # leaving the mesh is reported
    n, b, l = _march(olib, mesh, [1.5, 0, 0], 0.0, [1.0, 0, 0], 1.0, 1.0)
    assert n == -1


def test_comb_invariants(olib):
    """P14: count, multiplicity floor/ceil(M/N), monotone indices."""
    rng = np.random.default_rng(7)
    for N, M in [(1000, 1000), (1015, 1000), (640, 1000), (1, 7), (7, 1), (12345, 10000), (3, 10)]:
        for a in [2.0**-53, 0.5, 1 - 2.0**-53, float(rng.uniform())]:
            idx = (C.c_uint64 * M)()
            olib.oracle_comb_indices(N, M, a, idx)
            idx = np.array(idx[:], dtype=np.int64)
            assert len(idx) == M and idx.min() >= 0 and idx.max() <= N - 1
            assert np.all(np.diff(idx) >= 0)
            mult = np.bincount(idx, minlength=N)
            if a < 1 - 2.0**-20:   # (double)j + a rounds up to j+1 only for a within 2^-53*j of 1
                assert mult.min() >= M // N and mult.max() <= -(-M // N)
            # exact rational definition floor((j+a) N / M)
            from fractions import Fraction
            j = int(rng.integers(0, M))
            exact = int((Fraction(j) + Fraction(a)) * N / M)
            assert abs(int(idx[j]) - min(exact, N - 1)) <= 1


def test_flight_counter_limit_ends_the_particle_as_lost():
    """C.1: the flight counter is a 24-bit field of the Philox counter; a history that reaches 2^24 - 1
    flights under one id (a pure scatterer without census) ends as lost and the run reports it."""
    import mcdc_inputs as mi
    from oracle import Oracle
    o = Oracle(mi.infinite_medium(1.0, 1.0, 0.0, n_hist=1))
    with pytest.raises(RuntimeError, match="6"):
        o.run()
    c = o.counters(0)
    assert c["lost"] == 1 and c["flights"] == 1 << 24 and c["scatters"] == (1 << 24) - 1 and c["captures"] == 0
    assert c["segments"] == (1 << 24) - 1
