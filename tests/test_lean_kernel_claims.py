"""The claim behind `nearest_plane` of the lean pool kernels (csrc/mcdc_pool.cu): ranking the three
plane distances e_i / u_i by cross products, trusted only where the products differ by more than 2^-48 relative (and
numerators and directions agree in sign), picks the axis the DEFINITION picks — the smallest ROUNDED quotient, the
earlier axis on a tie (DESIGN.md section 3 C.5) — so that one division of the winner reproduces the three divisions.
Checked here in IEEE binary64 with numpy on random and on adversarial inputs (quotients equal or one ulp apart).  The
GPU side of the same claim is `test_plane_ranking_degenerate_starts` and every lean parity case."""
import numpy as np

EPS, TINY = 2.0 ** -48, 1e-290


def definition(e, u):
    """C.5: d_i = e_i / u_i clamped at 0, infinity for u_i = 0; first smallest."""
    with np.errstate(divide="ignore", invalid="ignore"):
        d = np.where(u == 0.0, np.inf, e / u)
    d = np.where(d < 0.0, 0.0, d)
    surf = np.zeros(d.shape[0], dtype=int)
    best = d[:, 0].copy()
    for a in (1, 2):
        lt = d[:, a] < best
        surf[lt] = a
        best = np.where(lt, d[:, a], best)
    return surf, best


def ranking(e, u):
    """The device code's decision, line by line: (sure, axis)."""
    sgn = np.signbit(e) != np.signbit(u)
    bad = sgn.any(axis=1)
    ae, au = np.abs(e), np.abs(u)
    with np.errstate(over="ignore", invalid="ignore"):
        pxy, pyx = ae[:, 0] * au[:, 1], ae[:, 1] * au[:, 0]
        d1 = pxy - pyx
        sure = np.abs(d1) > EPS * (pxy + pyx) + TINY
        yn = d1 > 0.0
        ew, uw = np.where(yn, ae[:, 1], ae[:, 0]), np.where(yn, au[:, 1], au[:, 0])
        pwz, pzw = ew * au[:, 2], ae[:, 2] * uw
        d2 = pwz - pzw
        sure &= np.abs(d2) > EPS * (pwz + pzw) + TINY
        zn = d2 > 0.0
    axis = np.where(zn, 2, np.where(yn, 1, 0))
    return sure & ~bad, axis


def _check(e, u):
    sure, axis = ranking(e, u)
    surf, best = definition(e, u)
    assert np.all(axis[sure] == surf[sure])
    rows = np.nonzero(sure)[0]
    with np.errstate(divide="ignore", invalid="ignore"):
        q = e[rows, axis[rows]] / u[rows, axis[rows]]
    assert np.all(q == best[rows])                     # the winner's own division IS the definition's minimum
    return sure.mean()


def test_random_flights_rank_like_the_definition():
    rng = np.random.default_rng(7)
    n = 2_000_000
    u = rng.normal(size=(n, 3)); u /= np.linalg.norm(u, axis=1)[:, None]
    lo = np.floor(rng.uniform(0, 63, size=(n, 3)))
    x = lo + rng.uniform(0, 1, size=(n, 3))
    x[: n // 10] = lo[: n // 10]                       # a tenth of them start exactly on their lower planes
    e = np.where(u > 0.0, lo + 1.0, lo) - x
    assert _check(e, u) > 0.85                          # and the fast path is the usual one


def test_ties_and_one_ulp_gaps_are_never_trusted_wrongly():
    rng = np.random.default_rng(11)
    n = 400_000
    # y is x scaled by a power of two (exactly equal quotients), or nudged by a few ulps on either side
    ex = rng.uniform(0.01, 1.0, n); ux = rng.uniform(0.01, 1.0, n)
    k = 2.0 ** rng.integers(-3, 4, n)
    ey, uy = ex * k, ux * k
    for _ in range(3):
        nudge = rng.integers(-3, 4, n)
        ey = np.where(nudge > 0, np.nextafter(ey, np.inf), np.where(nudge < 0, np.nextafter(ey, -np.inf), ey))
    ez = rng.uniform(0.01, 1.0, n); uz = rng.uniform(1e-3, 1.0, n)
    e = np.stack([ex, ey, ez], 1); u = np.stack([ux, uy, uz], 1)
    sign = rng.choice([-1.0, 1.0], size=(n, 3))
    _check(e * sign, u * sign)
    # permuted axes: the tie may sit between any two of them
    for perm in ((1, 2, 0), (2, 0, 1), (0, 2, 1)):
        _check((e * sign)[:, perm], (u * sign)[:, perm])


def test_degenerate_inputs_fall_back():
    e = np.array([[0.0, 0.0, 0.5], [0.3, 0.2, 0.1], [0.3, -0.2, 0.1], [1e-300, 1e-300, 1.0], [np.inf, 0.5, 0.5], [0.5, 0.5, 0.5]])
    u = np.array([[0.6, 0.8, 0.0], [0.0, 0.0, 1.0], [0.6, 0.7, 0.4], [1e-10, 1e-10, 1.0], [0.6, 0.7, 0.4], [0.0, 0.0, 1.0]])
    sure, axis = ranking(e, u)
    surf, _ = definition(e, u)
    # corner start, two zero cosines, a negative numerator, underflowing products, an infinite plane: not trusted —
    # unless the ranking is right anyway (an axis with u = 0 loses to a finite one by a wide margin)
    assert not sure[0] and not sure[2] and not sure[3] and not sure[4]
    assert np.all(axis[sure] == surf[sure])


def test_fp32_first_guess_of_the_group_transfer_is_confirmed_or_rejected_correctly():
    """Lean pool kernels, A9: the guess c = number of fp32 thresholds <= xi is taken only when the fp64 row confirms
    it (row[c] above xi or c = G - 1; row[c - 1] not above xi or c = 0); for a row that does not decrease this is the
    result of the definition's linear search (first j with xi < row[j], else G - 1), whatever the fp32 rounding did."""
    rng = np.random.default_rng(3)
    G = 7
    for trial in range(200):
        pdf = rng.uniform(0, 1, G) * (rng.uniform(0, 1, G) < 0.7)       # zeros: leading, trailing and inside
        if pdf.sum() == 0.0:
            pdf[rng.integers(0, G)] = 1.0
        run = np.cumsum(pdf); row = run / run[-1]; row[-1] = 1.0
        thr = np.full(8, np.inf, dtype=np.float32); thr[: G - 1] = row[: G - 1].astype(np.float32)
        xi = np.concatenate([rng.uniform(0, 1, 2000), row[:-1][row[:-1] > 0],                # (exactly on an entry)
                             np.nextafter(row[:-1], 0.0)[row[:-1] > 0], np.nextafter(row[:-1], 1.0)])
        xi = xi[(xi > 0.0) & (xi < 1.0)]
        lin = np.array([next((j for j in range(G - 1) if x < row[j]), G - 1) for x in xi])
        c = (xi.astype(np.float32)[:, None] >= thr[None, :7]).sum(1)
        ok = ((c == G - 1) | (xi < row[np.minimum(c, G - 1)])) & ((c == 0) | ~(xi < row[np.maximum(c - 1, 0)]))
        assert np.all(c[ok] == lin[ok])
        assert ok.mean() > 0.9
