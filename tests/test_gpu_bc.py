"""Non-periodic boundaries in k (cgks_fill_halo_bc).  The paper names its boundary types without
formulas, so the rules are DESIGN.md reading B1; what can be pinned is pinned:
  * slip wall = symmetry plane, by the method of images: a flow between two slip walls IS the upper half of a periodic flow
    on the doubled domain whose data are mirror-symmetric about the wall planes.  The CPU oracle (periodic only) runs the
    doubled domain; the library runs the half domain with CGKS_BC_SLIP_WALL on both sides; they must agree field by field.
    Every sign and index rule of the mirror image of Q, G and D is exercised (a wrong one is an O(1) error).
  * no-slip adiabatic wall, outflow, far field: invariants (no mass / energy flux through a wall, wall friction has the
    right sign, uniform flow preserved) -- parity unpinned."""
import numpy as np
import pytest

from paper_2508_08965_b200 import binding, inputs, slab
from tests import parity

pytestmark = pytest.mark.gpu


def _symmetric_channel(n=8, visc=True):
    """Doubled periodic box 2 x 2 x 4 with 2n planes in k, data mirror-symmetric about the planes k = 0 and k = n."""
    ni = nj = n; nk = 2 * n
    nodes = inputs.cartesian_nodes((ni, nj, nk), 0.0, 1.0)
    nodes[0] *= 2.0; nodes[1] *= 2.0; nodes[2] = nodes[2] * 4.0 - 2.0          # z in [-2, 2]: walls at z = 0 and z = +-2
    x, y, z = inputs.cell_centroids(nodes)
    cz = np.cos(np.pi * z / 2.0); sz = np.sin(np.pi * z / 2.0)                  # even / odd about both wall planes
    rho = 1.0 + 0.1 * cz * np.cos(np.pi * x) + 0.05 * np.cos(np.pi * z)
    u = 0.3 * np.sin(np.pi * x) * cz + 0.1
    v = -0.2 * np.cos(np.pi * y) * (1.0 + 0.5 * cz)
    w = 0.25 * sz * np.cos(np.pi * x) * np.cos(np.pi * y)
    p = 1.0 + 0.1 * cz * np.cos(np.pi * y)
    Q = inputs.prim_to_cons(rho, u, v, w, p)
    prm = inputs.tgv_params(Re=100.0) if visc else dict(inputs.sine_params(), tau_c1=0.05, tau_c2=5.0)
    return dict(nodes=nodes, Q=Q, G=None, D=None, params=prm, nonlinear=1, cfl=0.5)


def _half_domain(w, n):
    """Sub-domain context holding the upper half (planes n .. 2n-1) of the doubled box, halos to be filled by the walls."""
    s = binding.Solver(w["nodes"], binding.make_params(**w["params"], nonlinear=w["nonlinear"]), slab=(n, n))
    import torch
    s.set_state(slab.extended(torch.from_numpy(w["Q"]).to(s.device), n, n, 1))
    return s


@pytest.mark.parametrize("visc", [True, False])
def test_slip_walls_equal_the_symmetric_periodic_flow(visc):
    n = 8
    w = _symmetric_channel(n, visc)
    nsteps = 6
    orc, dts = parity.run_oracle(w, nsteps)
    # the oracle's flow stays mirror-symmetric (to round-off): the premise of the method of images
    assert np.abs(orc[0][0][n:] - orc[0][0][:n][::-1]).max() < 1e-12 and np.abs(orc[0][3][n:] + orc[0][3][:n][::-1]).max() < 1e-12
    s = _half_domain(w, n)
    for dt in dts:
        s.step_bounded(dt, binding.BC_SLIP_WALL, binding.BC_SLIP_WALL)
    s.status()
    Q, G, D = (t.cpu().numpy() for t in s.get_state()); s.close()
    gpu = (Q[:, 2:-2], G[:, :, 2:-2], D[:, :, 2:-2])
    ref = (orc[0][:, n:], orc[1][:, :, n:], orc[2][:, :, n:])
    half_nodes = w["nodes"][:, n:]
    errs = parity.field_errors(gpu, ref, half_nodes, w["Q"][:, n:])
    worst = max(errs, key=errs.get)
    assert errs[worst] <= nsteps * 1e-10, (worst, errs[worst])


@pytest.mark.parametrize("kind", [binding.BC_SLIP_WALL, binding.BC_NOSLIP_WALL])
def test_walls_pass_no_mass_and_no_energy(kind):
    """A slip wall is impermeable and adiabatic to round-off (the mirror image makes the mass and energy fluxes through the
    wall face vanish identically) and leaves the total tangential momentum unchanged.  The no-slip ghost state (all velocity
    components reversed at the mirrored position) does so only to first order: the reversed particles of the second-order
    kinetic solution start from tangentially displaced positions, which leaves a mass flux proportional to the tangential
    gradients (a property of the ghost-cell reading B1; 2e-5 of the mass over 10 steps here); the
    wall decelerates the tangential flow next to it."""
    n = 8
    w = _symmetric_channel(n, True)
    s = _half_domain(w, n)
    Q0 = s.get_state()[0][:, 2:-2].cpu().numpy()
    for _ in range(10):
        s.fill_halo_bc(0, kind); s.fill_halo_bc(1, kind)          # the CFL reduction reads owned planes only; halos for the stage
        s.step_bounded(s.compute_dt(0.4), kind, kind)
    s.status()
    Q1 = s.get_state()[0][:, 2:-2].cpu().numpy(); s.close()
    tot0, tot1 = Q0.sum(axis=(1, 2, 3)), Q1.sum(axis=(1, 2, 3))
    tol = 1e-13 if kind == binding.BC_SLIP_WALL else 1e-4
    assert abs(tot1[0] / tot0[0] - 1) < tol and abs(tot1[4] / tot0[4] - 1) < tol
    if kind == binding.BC_SLIP_WALL:
        assert abs(tot1[1] - tot0[1]) < 1e-11 * np.abs(Q0[1]).sum()
    else:
        assert tot1[1] < tot0[1] * (1 - 1e-4)                      # mean flow u = 0.1 + ... loses x-momentum to the walls


def test_far_field_and_outflow_preserve_a_uniform_flow_and_errors():
    n = 8
    nodes = inputs.cartesian_nodes(n, 0.0, 1.0)
    prm = binding.make_params(**inputs.tgv_params(Re=100.0), nonlinear=1)
    Qu = inputs.free_stream((n, n, n))
    import torch
    for kinds in ((binding.BC_FARFIELD, binding.BC_OUTFLOW), (binding.BC_OUTFLOW, binding.BC_FARFIELD)):
        s = binding.Solver(nodes, prm, slab=(0, n))
        s.set_state(slab.extended(torch.from_numpy(Qu), 0, n, 1))
        far = Qu[:, 0, 0, 0]
        for _ in range(5):
            dt = s.compute_dt(0.5)
            for stage in (1, 2):
                s.fill_halo_bc(0, kinds[0], far); s.fill_halo_bc(1, kinds[1], far)
                s.stage(stage, dt)
        Q, G, D = (t.cpu().numpy() for t in s.get_state())
        assert np.abs(Q[:, 2:-2] - Qu).max() < 1e-13 and np.abs(G[:, :, 2:-2]).max() < 1e-11 and np.abs(D[:, :, 2:-2]).max() < 1e-12
        with pytest.raises(binding.CgksError):
            s.fill_halo_bc(0, binding.BC_FARFIELD)                 # no state given
        with pytest.raises(binding.CgksError):
            s.fill_halo_bc(2, binding.BC_OUTFLOW)
        s.close()
    c = binding.Solver(inputs.curvilinear_nodes(n), prm, slab=(0, n))
    with pytest.raises(binding.CgksError):
        c.fill_halo_bc(0, binding.BC_SLIP_WALL)                    # uniform Cartesian meshes only
    c.close()
