"""Pins for the rigid-molecule oracle (oracle/md_oracle_rigid.c; R20).

The paper prints no equations for this extension, so every check is against something the mathematics fixes and that is
written here independently of the oracle: a numpy site-site energy and its numerical gradient (forces, torques), the
conservation laws of the free rigid rotor, orthonormality of the rotation matrix, time reversal, the dt^2 scaling of a
second-order symplectic scheme, and the closed-form precession of a free symmetric top."""
import math

import numpy as np
import pytest

from md_workloads import body_inertia, cross_body, random_rotations, rigid_state, tetrahedron_body
from md_workloads.configs import R_WCA
from oracle.md_oracle import OracleRigid


def np_energy(R, A, body, box, r_cut):
    """Site-site truncated, shifted LJ between sites of different molecules; plain numpy, minimum image by rounding."""
    nm, ns = R.shape[0], body.shape[0]
    s = (R[:, None, :] + np.einsum("mij,kj->mki", A, body)).reshape(nm * ns, 3)
    d = s[:, None, :] - s[None, :, :]
    d -= box * np.round(d / box)
    r = np.sqrt((d * d).sum(-1))
    mol = np.repeat(np.arange(nm), ns)
    mask = (mol[:, None] != mol[None, :]) & (r < r_cut)
    uc = 4.0 * (r_cut ** -12 - r_cut ** -6)
    with np.errstate(divide="ignore", invalid="ignore"):
        u = np.where(mask, 4.0 * (r ** -12 - r ** -6) - uc, 0.0)
    return 0.5 * u.sum()


def rot(axis, eps):
    """Rotation by eps about a unit axis (Rodrigues)."""
    k = np.asarray(axis, float)
    Kx = np.array([[0, -k[2], k[1]], [k[2], 0, -k[0]], [-k[1], k[0], 0]])
    return np.eye(3) + math.sin(eps) * Kx + (1 - math.cos(eps)) * (Kx @ Kx)


def dense_state(n_side=3, body=None, seed=5, density=0.22, T=1.0, jit=0.15):
    body = tetrahedron_body(0.9) if body is None else body
    R, A, V, pi, box = rigid_state(n_side ** 3, body, density, T, seed)
    rng = np.random.default_rng(seed)
    R = np.mod(R + rng.uniform(-jit, jit, R.shape), box)
    return body, R, A, V, pi, box


def test_r1_force_and_torque_are_minus_the_gradient_of_a_numpy_energy():
    for body in (tetrahedron_body(0.9), cross_body()):
        body, R, A, V, pi, box = dense_state(3, body, density=0.2)
        o = OracleRigid(R.shape[0], body, box, R_WCA, 0.4, 0.004)
        o.set_state(R, A, V, pi)
        F, T = o.force_torque()
        e = o.energies()
        assert e.pe == pytest.approx(np_energy(R, A, body, box, R_WCA), rel=1e-12)
        assert np.abs(F).max() > 1.0                                          # the state does interact
        assert np.abs(F.sum(0)).max() <= 1e-11 * np.abs(F).sum()              # zero net force
        h = 1e-5
        fscale = np.abs(F).max()
        for m in (0, 7, 13, 26):
            for c in range(3):
                Rp, Rm = R.copy(), R.copy()
                Rp[m, c] += h
                Rm[m, c] -= h
                g = (np_energy(Rp, A, body, box, R_WCA) - np_energy(Rm, A, body, box, R_WCA)) / (2 * h)
                assert abs(F[m, c] + g) <= 1e-7 * fscale
                ax = np.eye(3)[c]
                Ap, Am = A.copy(), A.copy()
                Ap[m] = rot(ax, h) @ A[m]
                Am[m] = rot(ax, -h) @ A[m]
                g = (np_energy(R, Ap, body, box, R_WCA) - np_energy(R, Am, body, box, R_WCA)) / (2 * h)
                assert abs(T[m, c] + g) <= 1e-7 * fscale                       # torque about the centre of mass, space frame


def test_r2_neighbor_sets_are_the_definition_and_exclude_the_own_molecule():
    body, R, A, V, pi, box = dense_state(4, density=0.25)
    o = OracleRigid(R.shape[0], body, box, R_WCA, 0.4, 0.004)
    o.set_state(R, A, V, pi)
    counts, flat = o.neighbors()
    s = o.sites()
    assert s.min() >= 0 and s.max() < box
    ns = body.shape[0]
    d = s[:, None, :] - s[None, :, :]
    d -= box * np.round(d / box)
    r2 = (d * d).sum(-1)
    mol = np.repeat(np.arange(R.shape[0]), ns)
    want = (r2 < (R_WCA + 0.4) ** 2) & (mol[:, None] != mol[None, :])
    off = np.concatenate([[0], np.cumsum(counts)])
    for i in range(len(counts)):
        assert np.array_equal(np.sort(flat[off[i]:off[i + 1]]), np.nonzero(want[i])[0])
    # sites sit where the rotation matrix puts them
    want_s = np.mod((R[:, None, :] + np.einsum("mij,kj->mki", A, body)).reshape(-1, 3), box)
    dd = s - want_s
    dd -= box * np.round(dd / box)
    assert np.abs(dd).max() < 1e-12


@pytest.mark.parametrize("body", [cross_body(), cross_body(0.6, 0.35, 0.35), tetrahedron_body(1.0)])
def test_r3_torque_free_top(body):
    """One molecule, nothing to interact with: the space-frame angular momentum A pi is conserved to rounding by every
    sub-rotation, the rotation matrix stays orthonormal, the rotational energy oscillates with an amplitude ~ dt^2
    (exactly conserved for a spherical top), and the centre of mass moves uniformly."""
    I = body_inertia(body)
    box = 50.0
    R0 = np.array([[25.0, 25.0, 25.0]])
    A0 = random_rotations(1, 11)
    V0 = np.array([[0.3, -0.2, 0.1]])
    pi0 = np.array([[0.9, -1.4, 0.6]]) * np.sqrt(I)
    amp = []
    for dt in (0.02, 0.01):
        o = OracleRigid(1, body, box, R_WCA, 0.4, dt)
        o.set_state(R0, A0, V0, pi0)
        e0 = o.energies()
        l0 = np.array([e0.lx, e0.ly, e0.lz])
        assert np.allclose(l0, A0[0] @ pi0[0], rtol=1e-14)
        assert e0.ke_rot == pytest.approx(0.5 * float((pi0[0] ** 2 / I).sum()), rel=1e-14)
        assert e0.ke_trans == pytest.approx(0.5 * body.shape[0] * float((V0 ** 2).sum()), rel=1e-14)
        dev = 0.0
        steps = int(round(8.0 / dt))
        for _ in range(steps // 20):
            o.step(20)
            e = o.energies()
            assert np.abs(np.array([e.lx, e.ly, e.lz]) - l0).max() <= 1e-12 * np.abs(l0).max()
            dev = max(dev, abs(e.ke_rot - e0.ke_rot) / e0.ke_rot)
        R, A, V, pi = o.state()
        assert np.abs(A[0] @ A[0].T - np.eye(3)).max() < 1e-12 and np.linalg.det(A[0]) == pytest.approx(1.0, abs=1e-12)
        assert np.allclose(R[0], R0[0] + V0[0] * dt * steps, atol=1e-10) and np.allclose(V, V0, atol=1e-15)
        assert float((pi[0] ** 2).sum()) == pytest.approx(float((pi0[0] ** 2).sum()), rel=1e-12)      # |pi| is conserved
        amp.append(dev)
    if np.ptp(I) < 1e-12:
        assert max(amp) < 1e-12                                                # spherical top: every sub-rotation conserves it
    else:
        assert 3.0 < amp[0] / amp[1] < 5.0                                     # second order: dt -> dt/2 quarters the error
        assert amp[1] < 1e-3


def test_r4_symmetric_top_precession_rate():
    """Free symmetric top (I1 = I2 != I3): pi_3 is constant and (pi_1, pi_2) turn at Omega = pi_3 (1/I3 - 1/I1)
    (textbook Euler equations).  The splitting reproduces the rate to O(dt^2)."""
    body = cross_body(0.6, 0.35, 0.35)            # moments: I1 = 2(b^2+c^2) != I2 = I3  -> symmetric about body x
    I = body_inertia(body)
    assert abs(I[1] - I[2]) < 1e-15 and abs(I[0] - I[1]) > 0.1
    dt, steps = 0.002, 2000
    o = OracleRigid(1, body, 40.0, R_WCA, 0.4, dt)
    pi0 = np.array([[0.8, 0.5, 0.0]])
    o.set_state(np.array([[20.0, 20.0, 20.0]]), np.eye(3)[None], np.zeros((1, 3)), pi0)
    o.step(steps)
    _, _, _, pi = o.state()
    assert pi[0, 0] == pytest.approx(0.8, rel=1e-6)          # constant for the exact flow; O(dt^2) for the splitting
    omega = 0.8 * (1.0 / I[0] - 1.0 / I[1])       # d pi_2/dt = (1/I1 - 1/I3) pi_1 pi_3 ... about the symmetry axis x
    ang = math.atan2(pi[0, 2], pi[0, 1])
    want = -omega * dt * steps
    diff = (ang - want + math.pi) % (2 * math.pi) - math.pi
    assert abs(diff) < 5e-4
    assert math.hypot(pi[0, 1], pi[0, 2]) == pytest.approx(0.5, rel=1e-6)
    assert float((pi[0] ** 2).sum()) == pytest.approx(0.8 ** 2 + 0.5 ** 2, rel=1e-13)      # |pi| exactly


def test_r5_reversibility_and_energy_scaling_of_an_interacting_system():
    body, R, A, V, pi, box = dense_state(3, density=0.12, T=1.0, jit=0.1)
    fl = []
    for dt in (0.004, 0.002):
        o = OracleRigid(R.shape[0], body, box, R_WCA, 0.4, dt)
        o.set_state(R, A, V, pi)
        e0 = o.energies()
        errs = []
        for _ in range(60):
            assert o.step(int(round(0.04 / dt))) == 0
            e = o.energies()
            errs.append(e.total - e0.total)
            assert max(abs(e.px), abs(e.py), abs(e.pz)) < 1e-11
        fl.append(np.std(errs))
        assert e.n_rebuilds >= 1 and e.pe > 0.0 and abs(e.ke - e0.ke) > 1e-3       # the molecules did collide
    assert 2.8 < fl[0] / fl[1] < 5.5                                             # dt^2
    assert fl[1] / R.shape[0] < 1e-4
    # reversal: n steps, flip V and pi, n steps
    o = OracleRigid(R.shape[0], body, box, R_WCA, 0.4, 0.004)
    o.set_state(R, A, V, pi)
    o.step(60)
    assert o.energies().n_rebuilds >= 1
    R1, A1, V1, pi1 = o.state()
    o.set_state(R1, A1, -V1, -pi1)
    o.step(60)
    R2, A2, V2, pi2 = o.state()
    d = R2 - R
    d -= box * np.round(d / box)
    assert np.abs(d).max() < 1e-9 and np.abs(A2 - A).max() < 1e-9 and np.abs(V2 + V).max() < 1e-9 and np.abs(pi2 + pi).max() < 1e-9


def test_r6_rebuild_rule_bound_counts_by_hand():
    """No interactions (far apart), one molecule moving and spinning: the speed bound |V| + |pi| b_max / I_min is constant,
    so the rebuild count after n steps is n // k0 with k0 the first k for which k dt bound > delta / 2."""
    body = tetrahedron_body(0.9)
    I = body_inertia(body)
    bmax = float(np.linalg.norm(body, axis=1).max())
    box, nm = 60.0, 8
    R = np.array([[7.5 + 15 * (m % 2), 7.5 + 15 * ((m // 2) % 2), 7.5 + 15 * (m // 4)] for m in range(nm)], float)
    A = random_rotations(nm, 3)
    V, pi = np.zeros((nm, 3)), np.zeros((nm, 3))
    V[5] = [1.2, -0.5, 0.3]
    pi[5] = [0.4, 0.1, -0.7]
    bound = float(np.linalg.norm(V[5]) + np.linalg.norm(pi[5]) / I.min() * bmax)
    dt, delta = 0.005, 0.4
    k0 = int(math.floor(0.5 * delta / (dt * bound))) + 1
    o = OracleRigid(nm, body, box, R_WCA, delta, dt)
    for steps in (k0 - 1, k0, 4 * k0 + 1):
        o.set_state(R, A, V, pi)
        o.step(steps)
        e = o.energies()
        assert e.n_rebuilds == steps // k0 and e.vbound == pytest.approx(bound, rel=1e-12) and e.pe == 0.0
