"""Pins of the oracle's sub-tile localisation (O9, reading R28: PAPER.md:361, 385) and of the real-time form of
the image-frequency branch (reading R29: PAPER.md:341, 453-467).  CPU only.

The paper names four interpolation schemes and prints no formula or worked example, so the pins are what the
mathematics fixes: the interpolation property, polynomial reproduction (closed forms), library routines that
implement the same named schemes (scipy's not-a-knot CubicSpline, its 'makima' Akima1DInterpolator, its linear
RegularGridInterpolator), the textbook Catmull-Rom form of Keys' kernel, brute force over the lattice, and the
symmetries of the rule.
"""
import numpy as np
import pytest
from scipy.interpolate import Akima1DInterpolator, CubicSpline, RegularGridInterpolator

import oracle
import synth

METHODS = [oracle.INTERP_BILINEAR, oracle.INTERP_BICUBIC, oracle.INTERP_SPLINE, oracle.INTERP_MAKIMA]
RNG = np.random.default_rng(28)


def _grid(Ty, Tx):
    return np.meshgrid(np.arange(Tx, dtype=np.float64), np.arange(Ty, dtype=np.float64))  # U (columns), V (rows)


def _pts(Ty, Tx, n=200):
    return RNG.uniform(0, Tx - 1, n), RNG.uniform(0, Ty - 1, n)


@pytest.mark.parametrize("method", METHODS)
@pytest.mark.parametrize("Ty,Tx", [(6, 7), (3, 3), (2, 5), (1, 4), (4, 1), (1, 1), (2, 2)])
def test_surface_passes_through_the_tile_centres(method, Ty, Tx):
    eta = RNG.normal(size=(Ty, Tx))
    U, V = _grid(Ty, Tx)
    got = oracle.interp_eval(eta, method, U, V).reshape(Ty, Tx)
    np.testing.assert_allclose(got, eta, rtol=0, atol=1e-13)


@pytest.mark.parametrize("method", METHODS)
@pytest.mark.parametrize("Ty,Tx", [(6, 7), (3, 4), (2, 5), (1, 4)])
def test_every_scheme_reproduces_a_plane(method, Ty, Tx):
    U, V = _grid(Ty, Tx)
    eta = 2.0 - 0.75 * U + 0.4 * V
    u, v = _pts(Ty, Tx)
    np.testing.assert_allclose(oracle.interp_eval(eta, method, u, v), 2.0 - 0.75 * u + 0.4 * v, atol=1e-12)


def test_bilinear_is_the_bilinear_form_and_matches_the_library():
    U, V = _grid(5, 6)
    eta = 1.0 + 0.5 * U - 0.25 * V + 0.125 * U * V  # exactly representable by the bilinear patch
    u, v = _pts(5, 6)
    np.testing.assert_allclose(oracle.interp_eval(eta, 0, u, v), 1.0 + 0.5 * u - 0.25 * v + 0.125 * u * v, atol=1e-13)
    eta = RNG.normal(size=(5, 6))
    lib = RegularGridInterpolator((np.arange(5.0), np.arange(6.0)), eta, method="linear")
    np.testing.assert_allclose(oracle.interp_eval(eta, 0, u, v), lib(np.stack([v, u], axis=1)), atol=1e-13)


@pytest.mark.parametrize("method", [oracle.INTERP_BICUBIC, oracle.INTERP_SPLINE])
@pytest.mark.parametrize("Ty,Tx", [(6, 7), (4, 4), (3, 5), (3, 3)])
def test_cubic_convolution_and_spline_reproduce_quadratics_up_to_the_border(method, Ty, Tx):
    """Keys' boundary samples and the not-a-knot conditions are exactly what makes this hold in the first and last
    interval too; a wrong boundary rule (replicated sample, natural spline) fails here."""
    U, V = _grid(Ty, Tx)
    f = lambda a, b: 1.0 + 0.3 * a - 0.2 * b + 0.05 * a * a - 0.07 * b * b + 0.02 * a * b
    u, v = _pts(Ty, Tx)
    np.testing.assert_allclose(oracle.interp_eval(f(U, V), method, u, v), f(u, v), atol=1e-12)


def test_spline_reproduces_cubics_and_matches_the_library_not_a_knot_spline():
    Ty, Tx = 6, 8
    U, V = _grid(Ty, Tx)
    f = lambda a, b: 0.5 - 0.1 * a ** 3 + 0.04 * b ** 3 + 0.3 * a * b * b - 0.2 * a * a + b
    u, v = _pts(Ty, Tx)
    np.testing.assert_allclose(oracle.interp_eval(f(U, V), 2, u, v), f(u, v), atol=1e-10)
    eta = RNG.normal(size=(Ty, Tx))
    got = oracle.interp_eval(eta, 2, u, v)
    for k in range(len(u)):  # rows first, then the column: the same separable order as R28
        col = CubicSpline(np.arange(Tx, dtype=float), eta, axis=1, bc_type="not-a-knot")(u[k])
        want = CubicSpline(np.arange(Ty, dtype=float), col, bc_type="not-a-knot")(v[k])
        assert abs(got[k] - want) <= 1e-12
    # three samples along an axis: the parabola through them
    eta3 = RNG.normal(size=(3, 3))
    got = oracle.interp_eval(eta3, 2, u[:50] * 2 / (Tx - 1), v[:50] * 2 / (Ty - 1))
    for k in range(50):
        uu, vv = u[k] * 2 / (Tx - 1), v[k] * 2 / (Ty - 1)
        col = [np.polyval(np.polyfit(np.arange(3.0), eta3[r], 2), uu) for r in range(3)]
        assert abs(got[k] - np.polyval(np.polyfit(np.arange(3.0), col, 2), vv)) <= 1e-12


def test_makima_matches_the_library_modified_akima():
    for (Ty, Tx) in [(6, 7), (3, 9), (5, 3), (4, 4)]:
        eta = RNG.normal(size=(Ty, Tx))
        eta[1, :] = eta[1, 0]  # a flat row: the w1 + w2 = 0 case of the slope rule
        u, v = _pts(Ty, Tx, 120)
        got = oracle.interp_eval(eta, 3, u, v)
        for k in range(len(u)):
            col = Akima1DInterpolator(np.arange(Tx, dtype=float), eta, axis=1, method="makima")(u[k])
            want = Akima1DInterpolator(np.arange(Ty, dtype=float), col, method="makima")(v[k])
            assert abs(got[k] - want) <= 1e-12


def test_cubic_convolution_interior_is_the_catmull_rom_polynomial():
    """Keys' a = -1/2 kernel on an interior interval is the Catmull-Rom cubic (textbook matrix form)."""
    f = RNG.normal(size=9)
    u = RNG.uniform(1.0, 7.0, 100)
    got = oracle.interp_eval(f[None, :], 1, u, 0 * u)
    i = np.floor(u).astype(int)
    t = u - i
    p0, p1, p2, p3 = f[i - 1], f[i], f[i + 1], f[i + 2]
    want = 0.5 * (2 * p1 + (-p0 + p2) * t + (2 * p0 - 5 * p1 + 4 * p2 - p3) * t ** 2 + (-p0 + 3 * p1 - 3 * p2 + p3) * t ** 3)
    np.testing.assert_allclose(got, want, atol=1e-13)


# ------------------------------------------------------------------------------------------
# the position rule
# ------------------------------------------------------------------------------------------
def _lattice_brute_force(eta, tile, t, method, r):
    """R28's search written with numpy: every lattice point inside the hull, first maximum in (j, i) order."""
    Ty, Tx = eta.shape
    ty, tx = divmod(int(t), Tx)
    half = tile * r
    ii = np.arange(-half, half + 1)
    u = tx + ii / half
    v = ty + ii / half
    ku, kv = (u >= 0) & (u <= Tx - 1), (v >= 0) & (v <= Ty - 1)
    UU, VV = np.meshgrid(u[ku], v[kv])
    val = oracle.interp_eval(eta, method, UU, VV).reshape(VV.shape)
    j, i = np.unravel_index(np.argmax(val), val.shape)  # numpy's argmax returns the first maximum in C order
    xc, yc = (tx + 0.5) * tile - 0.5, (ty + 0.5) * tile - 0.5
    return xc + ii[ku][i] / r, yc + ii[kv][j] / r, val[j, i]


@pytest.mark.parametrize("method", METHODS)
@pytest.mark.parametrize("tile,r", [(8, 1), (4, 3), (5, 2)])
def test_localise_is_the_first_maximum_over_the_lattice(method, tile, r):
    eta = RNG.normal(size=(6, 7))
    tiles = [0, 6, 3 * 7 + 3, 5 * 7, 5 * 7 + 6, 2 * 7 + 5]  # corners (clipped lattice), interior
    pos = oracle.localise(eta, tile, tiles, method, r)
    for k, t in enumerate(tiles):
        x, y, val = _lattice_brute_force(eta, tile, t, method, r)
        assert (pos.x[k], pos.y[k]) == (x, y) and pos.value[k] == val


@pytest.mark.parametrize("method", [oracle.INTERP_BICUBIC, oracle.INTERP_SPLINE])
def test_localise_finds_the_closed_form_peak_of_a_paraboloid(method):
    """eta = -(u-u0)^2 - (v-v0)^2 is reproduced exactly by both schemes, so the position is the lattice point nearest
    to the true peak, x0 = (u0 + 0.5) N_T - 0.5 (pixel centres at integers)."""
    tile, Ty, Tx = 32, 7, 9
    u0, v0 = 4.3, 2.6
    U, V = _grid(Ty, Tx)
    eta = 10.0 - (U - u0) ** 2 - (V - v0) ** 2
    x0, y0 = (u0 + 0.5) * tile - 0.5, (v0 + 0.5) * tile - 0.5  # 153.1, 98.7
    for (ty, tx) in [(3, 4), (2, 4), (3, 5), (2, 5)]:  # the four tiles around the peak all point at it
        xc, yc = (tx + 0.5) * tile - 0.5, (ty + 0.5) * tile - 0.5
        for r in (1, 4):
            pos = oracle.localise(eta, tile, [ty * Tx + tx], method, r)
            want_x = xc + np.round((x0 - xc) * r) / r
            want_y = yc + np.round((y0 - yc) * r) / r
            assert (pos.x[0], pos.y[0]) == (want_x, want_y)
            assert abs(pos.value[0] - (10.0 - ((want_x + 0.5) / tile - 0.5 - u0) ** 2
                                       - ((want_y + 0.5) / tile - 0.5 - v0) ** 2)) <= 1e-11


@pytest.mark.parametrize("method", METHODS)
def test_single_tile_and_single_row_grids(method):
    pos = oracle.localise(np.array([[3.0]]), 32, [0], method)
    assert (pos.x[0], pos.y[0], pos.value[0]) == (15.5, 15.5, 3.0)  # the tile centre (R18's tile, geometric centre)
    eta = np.array([[1.0, 5.0, 2.0, 0.5]])
    pos = oracle.localise(eta, 4, [1], method)
    assert pos.y[0] == 1.5 and 1.5 <= pos.x[0] <= 9.5 and pos.value[0] >= 5.0


@pytest.mark.parametrize("method", METHODS)
def test_whole_tile_shifts_move_the_position_by_the_tile_size(method):
    tile = 8
    core = np.zeros((9, 9))
    core[3:6, 3:6] = [[1.0, 2.0, 1.5], [2.5, 6.0, 4.0], [1.0, 3.0, 2.0]]
    a = np.zeros((12, 13))
    a[0:9, 0:9] = core
    b = np.zeros((12, 13))
    b[2:11, 3:12] = core  # shifted by 2 tile rows and 3 tile columns
    pa = oracle.localise(a, tile, [4 * 13 + 4], method, 2)
    pb = oracle.localise(b, tile, [6 * 13 + 7], method, 2)
    assert pb.x[0] == pa.x[0] + 3 * tile and pb.y[0] == pa.y[0] + 2 * tile
    # the three local schemes see the same neighbourhood; the spline is global (every sample reaches every point, with
    # a weight that decays about 0.27 per tile), so the distance to the border shows in the 4th digit of the value
    assert abs(pb.value[0] - pa.value[0]) <= (1e-3 if method == oracle.INTERP_SPLINE else 1e-12) * abs(pa.value[0])


@pytest.mark.parametrize("method", [oracle.INTERP_BILINEAR, oracle.INTERP_BICUBIC, oracle.INTERP_SPLINE])
def test_transposed_grid_gives_the_transposed_position(method):
    """The linear schemes are tensor products: the order of the two axes cannot matter (makima's slopes depend on the
    data, so its x-then-y order is part of the reading and is not symmetric)."""
    eta = RNG.normal(size=(6, 8))
    eta[2, 5] += 6.0
    p = oracle.localise(eta, 8, [2 * 8 + 5], method, 2)
    q = oracle.localise(np.ascontiguousarray(eta.T), 8, [5 * 6 + 2], method, 2)
    assert (p.x[0], p.y[0]) == (q.y[0], q.x[0]) and abs(p.value[0] - q.value[0]) <= 1e-12


def test_finer_lattice_contains_the_coarser_one():
    eta = RNG.normal(size=(5, 5))
    for m in METHODS:
        p1 = oracle.localise(eta, 6, [12], m, 1)
        p3 = oracle.localise(eta, 6, [12], m, 3)
        assert p3.value[0] >= p1.value[0]


def test_localise_rejects_bad_arguments():
    with pytest.raises(ValueError):
        oracle.localise(np.zeros((2, 2)), 8, [0], 4)
    with pytest.raises(ValueError):
        oracle.localise(np.zeros((2, 2)), 8, [0], 0, 0)


def test_a_source_between_two_tiles_is_placed_on_their_common_edge():
    """a pulsar on the boundary of two tiles contributes to both; equal contributions put the peak of
    every scheme half way between the two centres, i.e. on the common edge."""
    eta = np.full((5, 6), 0.1)
    eta[2, 2] = eta[2, 3] = 4.0
    for m in METHODS:
        p = oracle.localise(eta, 32, [2 * 6 + 2], m, 1)
        assert p.y[0] == 2 * 32 + 15.5
        if m == oracle.INTERP_BILINEAR:  # flat between the two centres: the first lattice point of the plateau
            assert p.x[0] == 2 * 32 + 15.5
        else:  # the cubics overshoot symmetrically: the maximum is in the middle
            assert p.x[0] == 3 * 32 - 0.5


# ------------------------------------------------------------------------------------------
# real-time form of the image-frequency branch (R29)
# ------------------------------------------------------------------------------------------
def test_realtime_frequency_equals_the_batch_branch_on_the_window():
    cfg = synth.scaled(synth.CONFIGS["imgfreq"], 128, 160, L=14).replace(n_transients=2, transient_peak=12.0, period=4)
    st, _ = synth.make_stack(cfg, device="cpu")
    st = st.numpy()
    st[5, 7, 9] = 300.0  # the running maximum jumps when snapshot 5 arrives
    window, tile, tau = 8, 16, 2.0
    Uw = window - 2
    rt = oracle.run_realtime_frequency(st, window, tile=tile, tau=tau)
    assert len(rt) == 12 and all(r is None for r in rt[:Uw - 1]) and all(r is not None for r in rt[Uw - 1:])
    for n in range(Uw - 1, 12):
        sub = st[n - Uw + 1:n + 3]
        batch = oracle.run(sub, tile=tile, tau=tau, branch=1)  # normalised by the window's own maximum
        Mn = max(float(st[:n + 3].max()), 1e-6)
        assert rt[n].res.M == Mn  # R24: everything seen so far
        assert (Mn == 300.0) == (n + 2 >= 5)
        scale = (batch.res.M / Mn) ** 2
        np.testing.assert_allclose(rt[n].eta, batch.eta * scale, rtol=1e-12)  # eta scales with 1 / M^2 ...
        np.testing.assert_allclose(rt[n].z, batch.z, rtol=1e-9, atol=1e-9)  # ... z (Eq. 11) does not
        assert np.array_equal(rt[n].kstar, batch.kstar)
        assert np.array_equal(rt[n].cands.tile, batch.cands.tile) and np.array_equal(rt[n].cands.snapshot, batch.cands.snapshot)
    assert sum(r.cands.n_found for r in rt[Uw - 1:]) > 0


def test_realtime_frequency_with_the_full_length_window_is_the_batch_result():
    st = synth.gaussian_noise_stack(9, 64, 64, seed=5).numpy()
    rt = oracle.run_realtime_frequency(st, 9, tile=16, tau=1.0, harmonics=2)
    batch = oracle.run(st, tile=16, tau=1.0, branch=1, harmonics=2)
    assert all(r is None for r in rt[:-1])
    np.testing.assert_array_equal(rt[-1].eta, batch.eta)  # M_n of the last unit is the batch M
    np.testing.assert_array_equal(rt[-1].z, batch.z)
    with pytest.raises(ValueError):
        oracle.run_realtime_frequency(st, 2)
