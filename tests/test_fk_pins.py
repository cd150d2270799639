"""Pins of the oracle's scene-graph update N12 (forward kinematics; PAPER.md:91,109 and
Table 5).  The paper prints no worked example, so the pins are what the mathematics fixes: the
definition's own sine / cosine against float64 and exact special values, closed forms computable by hand
(dyadic offsets, quarter turns about each axis, a prismatic joint, base yaw and position), random chains against
a float64 composition written here with numpy rotations, and the parent / child / held-object identities.
CPU only; the GPU parity test is tests/test_gpu_fk.py."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2306_07552_b200 import gen


def _T(x=0.0, y=0.0, z=0.0):
    return [1, 0, 0, x, 0, 1, 0, y, 0, 0, 1, z]


def _robot(parent, jt, axis, origin, cam_link=-1, mount=None, ee=-1):
    return gen.Robot(np.asarray(parent, np.int32), np.asarray(jt, np.int32), np.asarray(axis, np.float32),
                     np.asarray(origin, np.float32), cam_link, np.asarray(_T() if mount is None else mount, np.float32), ee)


def _m44(a):
    return np.asarray(a, np.float64).reshape(4, 4)


def test_sincos_against_float64_and_special_values(oracle_mod):
    x = np.concatenate([np.linspace(-50, 50, 400001), np.random.default_rng(3).uniform(-7, 7, 100000)]).astype(np.float32)
    s, c = oracle_mod.sincos(x)
    assert np.abs(s - np.sin(x.astype(np.float64))).max() < 2.5e-7
    assert np.abs(c - np.cos(x.astype(np.float64))).max() < 2.5e-7
    s0, c0 = oracle_mod.sincos(np.array([0.0, -0.0], np.float32))
    assert s0[0] == 0.0 and c0[0] == 1.0 and c0[1] == 1.0
    # odd / even symmetry is exact (every step of the definition is sign-symmetric)
    xs = np.abs(x[:1000])
    sp, cp = oracle_mod.sincos(xs)
    sm, cm = oracle_mod.sincos(-xs)
    assert np.array_equal(sp, -sm) and np.array_equal(cp, cm)
    # quadrants: a dropped sign or a swapped polynomial fails one of these
    q, _ = oracle_mod.sincos(np.array([np.pi / 2, np.pi, 3 * np.pi / 2, -np.pi / 2], np.float32))
    _, qc = oracle_mod.sincos(np.array([np.pi / 2, np.pi, 3 * np.pi / 2, 2 * np.pi], np.float32))
    assert np.allclose(q, [1, 0, -1, -1], atol=3e-7) and np.allclose(qc, [0, -1, 0, 1], atol=3e-7)


def test_zero_joints_dyadic_offsets_are_exact(oracle_mod):
    """All joints at 0, base at a dyadic position with yaw 0: every transform is a pure translation whose
    entries are sums of dyadic numbers -- exact in binary32 whatever the order."""
    r = _robot([-1, 0, 1, 1], [1, 2, 1, 0], [[0, 1, 0], [0, 1, 0], [1, 0, 0], [0, 0, 1]],
               [_T(0, 0.25, 0), _T(0.5, 0.5, 0), _T(0, 0.125, -0.75), _T(-0.25, 0, 1.0)], cam_link=2, mount=_T(0, 0.5, 0.0625), ee=3)
    base = np.array([[3.0, -2.5, 0.0]], np.float32)
    cam, xf = oracle_mod.fk(r, base, np.zeros((1, 4), np.float32), 6, 1, held_slot=np.array([5], np.int32),
                            held_xform=np.array([_T(0.0, -0.125, 0.0)], np.float32))
    exp = {1: (3.0, 0.25, -2.5), 2: (3.5, 0.75, -2.5), 3: (3.5, 0.875, -3.25), 4: (3.25, 0.75, -1.5)}
    for slot, t in exp.items():
        assert np.array_equal(_m44(xf[0, slot]), np.array([[1, 0, 0, t[0]], [0, 1, 0, t[1]], [0, 0, 1, t[2]], [0, 0, 0, 1.0]])), slot
    assert np.array_equal(_m44(cam[0])[:3, 3], [3.5, 1.375, -3.1875])           # link 2 + mount
    assert np.array_equal(_m44(xf[0, 5])[:3, 3], [3.25, 0.625, -1.5])           # held object: link 3 + offset
    assert np.array_equal(xf[0, 0], np.zeros(16, np.float32))                   # slots outside the robot are left alone


@pytest.mark.parametrize("axis,src,dst", [((0, 1, 0), (1, 0, 0), (0, 0, -1)), ((0, 1, 0), (0, 0, 1), (1, 0, 0)),
                                          ((1, 0, 0), (0, 1, 0), (0, 0, 1)), ((1, 0, 0), (0, 0, 1), (0, -1, 0)),
                                          ((0, 0, 1), (1, 0, 0), (0, 1, 0)), ((0, 0, 1), (0, 1, 0), (-1, 0, 0))])
def test_quarter_turn_is_right_handed(oracle_mod, axis, src, dst):
    """A revolute joint at +90 degrees about a coordinate axis maps the basis vectors as a right-handed rotation
    does (x -> y about z, y -> z about x, z -> x about y): fixes the sign of every sine term of N12b."""
    r = _robot([-1], [1], [axis], [_T()])
    _, xf = oracle_mod.fk(r, np.zeros((1, 3), np.float32), np.array([[np.pi / 2]], np.float32), 1, 0)
    R = _m44(xf[0, 0])[:3, :3]
    assert np.allclose(R @ np.array(src, np.float64), dst, atol=3e-7)
    assert np.allclose(R @ np.array(axis, np.float64), axis, atol=3e-7)          # the axis is fixed


def test_prismatic_and_base_yaw_closed_forms(oracle_mod):
    # prismatic: translation theta * axis, exact for dyadic values
    r = _robot([-1], [2], [[0, 1, 0]], [_T(0.5, 0, 0)])
    _, xf = oracle_mod.fk(r, np.zeros((1, 3), np.float32), np.array([[0.375]], np.float32), 1, 0)
    assert np.array_equal(_m44(xf[0, 0]), np.array([[1, 0, 0, 0.5], [0, 1, 0, 0.375], [0, 0, 1, 0], [0, 0, 0, 1.0]]))
    # base: yaw turns about +Y (a robot facing -Z turns to face -X at +90 degrees), position is (x, 0, z)
    r = _robot([-1], [0], [[0, 1, 0]], [_T(0, 0, -1.0)], cam_link=-1, mount=_T(0, 1.25, 0))
    cam, xf = oracle_mod.fk(r, np.array([[2.0, 5.0, np.pi / 2]], np.float32), np.zeros((1, 1), np.float32), 1, 0)
    assert np.allclose(_m44(xf[0, 0])[:3, 3], [1.0, 0.0, 5.0], atol=1e-6)       # one metre ahead of the base, now along -X
    assert np.allclose(_m44(cam[0])[:3, 3], [2.0, 1.25, 5.0], atol=1e-6)
    assert np.allclose(_m44(cam[0])[:3, :3] @ [0, 0, -1.0], [-1, 0, 0], atol=3e-7)


def _rot64(axis, th):
    a = np.asarray(axis, np.float64)
    Kx = np.array([[0, -a[2], a[1]], [a[2], 0, -a[0]], [-a[1], a[0], 0]])
    return np.eye(3) + np.sin(th) * Kx + (1 - np.cos(th)) * (Kx @ Kx)           # Rodrigues, the other textbook form


def test_random_chains_against_float64(oracle_mod):
    rng = np.random.default_rng(12)
    for trial in range(20):
        L = int(rng.integers(1, 12))
        parent = [-1] + [int(rng.integers(-1, l)) for l in range(1, L)]
        jt = rng.integers(0, 3, L)
        axis = rng.normal(size=(L, 3))
        axis /= np.linalg.norm(axis, axis=1, keepdims=True)
        origin = np.zeros((L, 3, 4))
        for l in range(L):
            origin[l, :, :3] = _rot64(rng.normal(size=3) / 1.7, rng.uniform(-3, 3)) if rng.uniform() < 0.7 else np.eye(3)
            ax = origin[l, :, :3]
            u, _, vt = np.linalg.svd(ax)
            origin[l, :, :3] = u @ vt
            origin[l, :, 3] = rng.uniform(-0.5, 0.5, 3)
        cam_link, ee = int(rng.integers(-1, L)), int(rng.integers(-1, L))
        mount = np.concatenate([_rot64([1, 0, 0], -0.3), [[0.1], [0.2], [-0.05]]], axis=1)
        r = _robot(parent, jt, axis, origin.reshape(L, 12), cam_link, mount.reshape(12), ee)
        N, K, slot0 = 5, L + 3, 2
        base = np.stack([rng.uniform(-5, 5, N), rng.uniform(-5, 5, N), rng.uniform(-6, 6, N)], axis=1).astype(np.float32)
        th = rng.uniform(-3, 3, (N, L)).astype(np.float32)
        held = np.array([-1, 0, K - 1, -1, 1], np.int32)
        hx = np.tile(np.concatenate([_rot64([0, 0, 1], 0.4), [[0.0], [0.01], [-0.1]]], axis=1).reshape(12), (N, 1)).astype(np.float32)
        cam, xf = oracle_mod.fk(r, base, th, K, slot0, held_slot=held, held_xform=hx)
        a32, o32 = axis.astype(np.float32).astype(np.float64), origin.reshape(L, 12).astype(np.float32).astype(np.float64).reshape(L, 3, 4)
        for n in range(N):
            def h(m34):
                return np.vstack([m34, [0, 0, 0, 1.0]])
            yaw = float(base[n, 2])
            B = np.eye(4)
            B[:3, :3] = _rot64([0, 1, 0], yaw)
            B[:3, 3] = [base[n, 0], 0, base[n, 1]]
            Wm = [B]
            for l in range(L):
                J = np.eye(4)
                if jt[l] == 1:
                    J[:3, :3] = _rot64(a32[l], float(th[n, l]))
                elif jt[l] == 2:
                    J[:3, 3] = float(th[n, l]) * a32[l]
                Wm.append(Wm[parent[l] + 1] @ h(o32[l]) @ J)
                if held[n] != slot0 + l:
                    assert np.allclose(_m44(xf[n, slot0 + l]), Wm[-1], atol=2e-5), (trial, n, l)
            assert np.allclose(_m44(cam[n]), Wm[cam_link + 1] @ h(mount.astype(np.float32).astype(np.float64)), atol=2e-5)
            if held[n] >= 0:
                assert np.allclose(_m44(xf[n, held[n]]), Wm[ee + 1] @ h(hx[n].astype(np.float64).reshape(3, 4)), atol=2e-5)
            assert np.array_equal(xf[n, :, 12:], np.tile([0, 0, 0, 1.0], (K, 1)) * (np.abs(xf[n]).sum(axis=1, keepdims=True) > 0))


def test_rotations_stay_orthonormal_and_children_follow_parents(oracle_mod):
    r = gen.robot_proxy()
    base, th, held, hx = gen.robot_states(r, 64, seed=1)
    K, slot0 = 25, 20
    cam, xf = oracle_mod.fk(r, base, th, K, slot0, held_slot=held, held_xform=hx)
    for n in range(64):
        for l in range(5):
            R = _m44(xf[n, slot0 + l])[:3, :3]
            assert np.allclose(R @ R.T, np.eye(3), atol=2e-6) and abs(np.linalg.det(R) - 1) < 2e-6
        # the camera rides on the torso: its height follows the lift joint exactly as the closed form says
        assert abs(_m44(cam[n])[1, 3] - (0.25 + 0.45 + float(th[n, 1]) + 0.5)) < 1e-6
        # moving only the last joint leaves every other link where it was
    th2 = th.copy()
    th2[:, 4] += 0.5
    cam2, xf2 = oracle_mod.fk(r, base, th2, K, slot0, held_slot=held, held_xform=hx)
    assert np.array_equal(xf[:, slot0:slot0 + 4], xf2[:, slot0:slot0 + 4]) and np.array_equal(cam, cam2)
    assert not np.array_equal(xf[:, slot0 + 4], xf2[:, slot0 + 4])


def test_bad_arguments(oracle_mod):
    r = _robot([0], [0], [[0, 1, 0]], [_T()])          # a link that is its own parent
    with pytest.raises(ValueError):
        oracle_mod.fk(r, np.zeros((1, 3), np.float32), np.zeros((1, 1), np.float32), 1, 0)
    r = _robot([-1], [0], [[0, 1, 0]], [_T()])
    with pytest.raises(ValueError):
        oracle_mod.fk(r, np.zeros((1, 3), np.float32), np.zeros((1, 1), np.float32), 1, 1)   # link slot outside K
