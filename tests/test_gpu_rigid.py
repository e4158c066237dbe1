"""GPU parity of the rigid-molecule path (md_set_rigid; R20) against the rigid oracle
(oracle/md_oracle_rigid.c) on the same seeded inputs.  Tolerances are north_star's: neighbor sets of the sites exact, site
forces 1e-10, positions (centres of mass, sites) after 10 steps 1e-9, energies 1e-9 relative; the rotation matrices and
momenta are compared at the same level."""
import numpy as np
import pytest

from md_workloads import cross_body, rigid_state, tetrahedron_body
from md_workloads.configs import R_WCA
from oracle.md_oracle import OracleRigid
from parity_util import ENERGY_RTOL, FORCE_RTOL, POS_ATOL, force_rel_err, pos_err, sets_equal

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def md():
    import paper_2003_14061_b200 as m
    m.load_library()
    return m


CASES = {
    # four slightly overlapping SP spheres at the corners of a tetrahedron, 1000 and 4096 molecules
    "tetra_1000": (10, tetrahedron_body(0.9), 0.12),
    "tetra_4096": (16, tetrahedron_body(0.9), 0.10),
    "cross_729": (9, cross_body(), 0.10),                      # asymmetric top, 6 sites; 4374 sites: a ragged tail
}


def make_pair(md, case, seed, jit=0.12, dt=0.004, **kw):
    n_side, body, rho = CASES[case]
    R, A, V, pi, box = rigid_state(n_side ** 3, body, rho, 1.0, seed)
    rng = np.random.default_rng(seed)
    R = np.mod(R + rng.uniform(-jit, jit, R.shape), box)
    nm, ns = R.shape[0], body.shape[0]
    o = OracleRigid(nm, body, box, R_WCA, 0.4, dt)
    o.set_state(R, A, V, pi)
    g = md.MDSystem(nm * ns, R_WCA, 0.4, dt, box=box, lattice="none", **kw)
    g.set_rigid(body)
    g.set_rigid_state(R, A, V, pi)
    return g, o, box, (R, A, V, pi), body


class _Sets:
    def __init__(self, o):
        self.o = o

    def neighbors(self):
        return self.o.neighbors()


@pytest.mark.parametrize("case", list(CASES))
def test_rigid_sets_forces_energies(md, case):
    for seed in (1, 2, 3):
        g, o, box, state, body = make_pair(md, case, seed)
        counts, lst = g.neighbors()
        nbad, first = sets_equal(counts, lst, _Sets(o))
        assert nbad == 0, f"site neighbor sets differ for {nbad} sites (first: site {first})"
        assert pos_err(g.positions(), o.sites(), box) <= 1e-12
        fo = o.site_forces()
        assert np.abs(fo).max() > 1.0
        assert force_rel_err(g.forces(), fo) <= FORCE_RTOL
        eg, eo = g.energies(), o.energies()
        assert eg.pe_pair == pytest.approx(eo.pe, rel=ENERGY_RTOL, abs=1e-9)
        assert eg.virial == pytest.approx(eo.virial, rel=ENERGY_RTOL, abs=1e-7)
        assert eg.ke == pytest.approx(eo.ke, rel=1e-12)                         # translational + rotational, from the site velocities
        for a, b in ((eg.px, eo.px), (eg.py, eo.py), (eg.pz, eo.pz)):
            assert abs(a - b) <= 1e-10
        assert eg.mean_neighbors == pytest.approx(eo.mean_neighbors, rel=1e-12) and eg.max_neighbors == eo.max_neighbors
        g.close()


@pytest.mark.parametrize("case", list(CASES))
@pytest.mark.parametrize("flags", [0, 2])
def test_rigid_ten_steps(md, case, flags):
    for seed in (1, 2):
        g, o, box, state, body = make_pair(md, case, seed, flags=flags)
        g.step(10)
        assert o.step(10) == 0
        Rg, Ag, Vg, pg = g.rigid_state()
        Ro, Ao, Vo, po = o.state()
        assert pos_err(Rg, Ro, box) <= POS_ATOL
        assert np.abs(Ag - Ao).max() <= 1e-9 and np.abs(Vg - Vo).max() <= 1e-8 and np.abs(pg - po).max() <= 1e-8
        assert np.abs(np.einsum("mij,mkj->mik", Ag, Ag) - np.eye(3)).max() < 1e-12
        assert pos_err(g.positions(), o.sites(), box) <= POS_ATOL
        eg, eo = g.energies(), o.energies()
        assert eg.ke == pytest.approx(eo.ke, rel=ENERGY_RTOL) and eg.pe == pytest.approx(eo.pe, rel=ENERGY_RTOL)
        assert eg.step == eo.step == 10 and eg.n_rebuilds == eo.n_rebuilds
        assert force_rel_err(g.forces(), o.site_forces()) <= 1e-8
        g.close()


def test_rigid_long_run_conserves_and_rebuilds(md):
    """400 steps with ~25 rebuilds: the site list must stay valid across re-sorts and periodic wraps (image offsets of the
    sites), so the energy is conserved as the oracle conserves it and momentum stays zero."""
    g, o, box, state, body = make_pair(md, "tetra_1000", 5)
    e0 = g.energies()
    g.step(400)
    o.step(400)
    eg, eo = g.energies(), o.energies()
    nm = state[0].shape[0]
    assert eg.n_rebuilds > 10 and abs(eg.n_rebuilds - eo.n_rebuilds) <= 1
    assert abs(eg.total - e0.total) / nm < 5e-3
    assert eg.total == pytest.approx(eo.total, rel=1e-6)
    assert max(abs(eg.px), abs(eg.py), abs(eg.pz)) < 1e-9
    # the sites are where the molecule state says they are, modulo the box
    R, A, V, pi = g.rigid_state()
    want = (R[:, None, :] + np.einsum("mij,kj->mki", A, body)).reshape(-1, 3)
    assert pos_err(g.positions(), want, box) <= 1e-11
    s = g.positions()
    assert s.min() >= 0.0 and s.max() < box


def test_rigid_rejects_bad_input(md):
    body = tetrahedron_body(0.9)
    g = md.MDSystem(4000, R_WCA, 0.4, 0.004, density=0.4, lattice="none")
    with pytest.raises(md.MDError):
        g.set_rigid(body + 0.1)                       # centre of mass not at the origin
    with pytest.raises(md.MDError):
        g.set_rigid(np.array([[0.5, 0, 0], [-0.5, 0, 0], [0.0, 0, 0]]))      # collinear: a zero moment
    with pytest.raises(md.MDError):
        g.set_rigid(cross_body()[[0, 1, 2, 3, 4]])    # 5 sites: 4000 is a multiple, but the frame is not principal / centred
    g.set_rigid(body)
    with pytest.raises(md.MDError):
        g.set_state(np.zeros((4000, 3)))              # rigid systems take molecule states
    g.close()
    g = md.MDSystem(4000, R_WCA, 0.4, 0.004, density=0.4, lattice="none", precision="f32")
    with pytest.raises(md.MDError):
        g.set_rigid(body)
    g.close()
