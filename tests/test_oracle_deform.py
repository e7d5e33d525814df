"""Pins for oracle steps O1/O2 (forward deformation, fp64) and O7 (inverse, fp32).

None of these re-types the oracle's formula: they use printed values, the identity pose,
the inverse round trip and the geometric properties that DEFINE a twist about +y and a
circular-arc bend about z (BASELINE.json configs B:7, B:8).
"""
import math

import numpy as np
import pytest

from conftest import read_golden

POSES = [(1.0, 0.0), (0.0, 0.8), (math.pi, 1.2), (0.7, 0.5), (1.3, 0.02755911)]


def _points(n, k, seed):
    rng = np.random.default_rng(seed)
    p = rng.uniform(-1.0, 1.0, size=(n, 3))
    if k > 0:                                  # stay clear of the fold-over k*y >= 1 (R7)
        p[:, 1] = np.minimum(p[:, 1], 0.8 / k if 0.8 / k < 1 else 1.0)
    return p


def test_worked_values(oracle):
    # SURVEY.md:397 worked values (fp64, computed independently of oracle/)
    for row in read_golden("deform_worked.txt"):
        th, k, x, y, z, X, Y, Z = map(float, row)
        got = oracle.forward_f64(th, k, [[x, y, z]])[0]
        np.testing.assert_allclose(got, [X, Y, Z], rtol=0, atol=2e-13)


def test_identity_pose_lattice_is_rest_lattice_bit_for_bit(oracle):
    # BASELINE.json:5 "the zero-deformation pose makes the rest/deformed mapping the identity"
    for nv in (8, 16, 12):
        lat = oracle.deform_lattice(nv, 0.0, 0.0).reshape(nv + 1, nv + 1, nv + 1, 3)
        c = ((2.0 * np.arange(nv + 1) - nv) / nv).astype(np.float32)
        assert np.array_equal(lat[..., 0], np.broadcast_to(c[None, None, :], lat.shape[:3]))
        assert np.array_equal(lat[..., 1], np.broadcast_to(c[None, :, None], lat.shape[:3]))
        assert np.array_equal(lat[..., 2], np.broadcast_to(c[:, None, None], lat.shape[:3]))


def test_identity_pose_inverse_is_identity(oracle):
    P = np.random.default_rng(0).uniform(-1, 1, size=(1000, 3)).astype(np.float32)
    assert np.array_equal(oracle.inverse_f32(0.0, 0.0, P), P)


def test_tiny_curvature_is_identity(oracle):
    p = _points(100, 0, 1)
    assert np.array_equal(oracle.forward_f64(0.0, 5e-7, p), p)


@pytest.mark.parametrize("pose", POSES)
def test_inverse_of_forward_is_identity(oracle, pose):
    # BASELINE.json:5 "inverse(forward(x)) returns x within 1e-6": fp64 forward, rounded once
    # to fp32 (as the lattice is), fp32 inverse.
    th, k = pose
    p = _points(100_000, k, 2)
    P = oracle.forward_f64(th, k, p).astype(np.float32)
    back = oracle.inverse_f32(th, k, P)
    err = np.abs(back.astype(np.float64) - p).max()
    assert err <= 1e-6, err


@pytest.mark.parametrize("theta", [1.0, 0.3, math.pi])
def test_twist_is_a_rotation_about_y_by_theta_of_y(oracle, theta):
    # definition (B:7): rotation about +y by theta_max*(y+1)/2: keeps y and the distance to the
    # y-axis, and turns the azimuth of every point by exactly that angle.
    p = _points(2000, 0, 3)
    q = oracle.forward_f64(theta, 0.0, p)
    np.testing.assert_allclose(q[:, 1], p[:, 1], rtol=0, atol=0)
    np.testing.assert_allclose(np.hypot(q[:, 0], q[:, 2]), np.hypot(p[:, 0], p[:, 2]), atol=1e-15)
    # rotation about +y by angle a maps the +z axis towards +x (right-handed): azimuth measured
    # as atan2(x, z) increases by a
    az0 = np.arctan2(p[:, 0], p[:, 2]); az1 = np.arctan2(q[:, 0], q[:, 2])
    a = theta * (p[:, 1] + 1.0) / 2.0
    diff = np.angle(np.exp(1j * (az1 - az0 - a)))
    assert np.abs(diff).max() < 1e-12
    # y = -1 is the fixed end of the twist
    fixed = np.array([[0.3, -1.0, -0.2]])
    np.testing.assert_allclose(oracle.forward_f64(theta, 0.0, fixed), fixed, atol=1e-16)


@pytest.mark.parametrize("k", [0.8, 1.2, 0.1])
def test_bend_is_a_circular_arc_about_z(oracle, k):
    # definition (B:8 "closed-form circular arc; the inverse is the arc-length unroll"):
    # the line {y = y0} maps to the circle of radius 1/k - y0 centred at (0, 1/k); the arc
    # length along the neutral fibre y = 0 is preserved (angle = k*x); z is untouched.
    p = _points(2000, k, 4)
    q = oracle.forward_f64(0.0, k, p)
    np.testing.assert_allclose(q[:, 2], p[:, 2], atol=0)
    rad = np.hypot(q[:, 0], q[:, 1] - 1.0 / k)
    np.testing.assert_allclose(rad, 1.0 / k - p[:, 1], atol=1e-13)
    ang = np.arctan2(q[:, 0], 1.0 / k - q[:, 1])          # angle from the downward radius
    np.testing.assert_allclose(ang, k * p[:, 0], atol=1e-12)
    # x = 0 is the fixed plane of the bend
    fixed = np.array([[0.0, 0.37, -0.5]])
    np.testing.assert_allclose(oracle.forward_f64(0.0, k, fixed), fixed, atol=1e-16)


def test_composite_is_bend_after_twist(oracle):
    # B:9, B:11 "a twist ... followed by a bend"
    p = _points(500, 1.2, 5)
    a = oracle.forward_f64(0.0, 1.2, oracle.forward_f64(math.pi, 0.0, p))
    b = oracle.forward_f64(math.pi, 1.2, p)
    np.testing.assert_allclose(a, b, atol=1e-15)


def test_lattice_is_forward_of_rest_lattice_rounded_once(oracle):
    nv, th, k = 8, 0.9, 0.6
    lat = oracle.deform_lattice(nv, th, k)
    c = (2.0 * np.arange(nv + 1) - nv) / nv
    zz, yy, xx = np.meshgrid(c, c, c, indexing="ij")        # x fastest
    rest = np.stack([xx, yy, zz], -1).reshape(-1, 3)
    # the float pose parameters are widened exactly to double
    want = oracle.forward_f64(np.float32(th), np.float32(k), rest).astype(np.float32)
    assert np.array_equal(lat, want)


# ---- O2x: the lattice is the CORRECTLY ROUNDED fp32 value of the closed form (R28) ----
def _mp_round_f32(v):
    """nearest float32 to the mpmath number v, decided in mpmath arithmetic (no double rounding)"""
    import mpmath as mp
    f = np.float32(float(v))
    cands = [f, np.nextafter(f, np.float32(-np.inf)), np.nextafter(f, np.float32(np.inf))]
    return min(cands, key=lambda c: abs(mp.mpf(float(c)) - v))


def _mp_forward(th, k, p):
    """the closed form of B:7/B:8 (twist about +y, circular-arc bend about z) at 60 digits, in the
    textbook arc form X = (1/k - y) sin(kx), Y = 1/k - (1/k - y) cos(kx) -- not the oracle's
    cancellation-free rearrangement"""
    import mpmath as mp
    mp.mp.dps = 60
    th, k = mp.mpf(float(np.float32(th))), mp.mpf(float(np.float32(k)))
    x, y, z = (mp.mpf(float(c)) for c in p)
    a = th * (y + 1) / 2
    tx, ty, tz = x * mp.cos(a) + z * mp.sin(a), y, -x * mp.sin(a) + z * mp.cos(a)
    if abs(k) < mp.mpf("1e-6"):
        return tx, ty, tz
    R = 1 / k
    return (R - ty) * mp.sin(k * tx), R - (R - ty) * mp.cos(k * tx), tz


@pytest.mark.parametrize("pose", POSES)
def test_exact_forward_is_the_correctly_rounded_closed_form(oracle, pose):
    th, k = pose
    p = _points(300, k, 5)
    got = oracle.forward_exact_f32(th, k, p)
    for i in range(len(p)):
        want = [_mp_round_f32(v) for v in _mp_forward(th, k, p[i])]
        assert [float(g) for g in got[i]] == [float(w) for w in want], (i, p[i])


@pytest.mark.parametrize("nv,pose", [(16, (1.0, 0.0)), (12, (0.7, 0.5)), (32, (math.pi, 1.2)), (24, (1.3, 0.02755911))])
def test_lattice_equals_exact_forward_on_every_point(oracle, nv, pose):
    # the fp64 fast path with its binary128 fallback must give the definition's bits everywhere
    lat, n_exact = oracle.deform_lattice(nv, *pose, count_exact=True)
    g = (2.0 * np.arange(nv + 1) - nv) / nv
    z, y, x = np.meshgrid(g, g, g, indexing="ij")
    p = np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1)
    want = oracle.forward_exact_f32(pose[0], pose[1], p)
    assert np.array_equal(lat.view(np.int32), want.view(np.int32))
    assert n_exact < 0.15 * len(p)            # the fallback is the exception (exact zeros such as the y = 0 plane, near-midpoint values)


def test_fp64_rounding_alone_is_not_the_definition(oracle):
    # why O2x exists: plain fp64 evaluation rounded to fp32 differs from the correctly rounded value on a
    # few entries of a large lattice, or at least needs the fallback there
    lat, n_exact = oracle.deform_lattice(64, 0.0, 0.8, count_exact=True)
    assert n_exact > 0
