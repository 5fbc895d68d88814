"""-m gpu parity of the Davidson step / solve: ground energies against dense eigh of the oracle's
H_eff (BASELINE.json: |θ − E_ref| ≤ 1e-9, reading r13) and step-by-step against oracle/davidson.py."""
import numpy as np
import pytest

import workloads as wlmod
from oracle import heff, davidson, lattice, dmrg, export
from _gpu import device_problem, config1_problem, TOL_ENERGY

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def check_energy(pb, m_max=16, tol=1e-9):
    H = heff.dense_heff(pb)
    assert np.abs(H - H.T).max() <= 1e-12 * np.abs(H).max()
    E = np.linalg.eigvalsh(H)[0]
    dp = device_problem(pb)
    dav = dp.davidson(m_max=m_max, tol=tol, max_iter=2000)
    dav.start(dp.psi_from_host(pb.psi))
    x = dp.new_vector()
    theta, rn, n_apply, ok = dav.solve(x)
    assert ok and rn <= tol
    assert abs(theta - E) <= TOL_ENERGY * max(1.0, abs(E))
    # the Ritz vector really is an eigenvector: ‖Hx − θx‖ ≤ tol, ‖x‖ = 1
    xv = heff.psi_to_vec(pb, dp.to_blocks(x))
    assert abs(np.linalg.norm(xv) - 1.0) <= 1e-12
    assert np.linalg.norm(H @ xv - theta * xv) <= 10 * tol
    return dp, theta, n_apply


def test_energy_small_spinless():
    pb = heff.problem_from_workload(wlmod.lattice_workload("spinless", 5, 24, seed=3))
    check_energy(pb)


def test_energy_small_hubbard_with_restarts():
    thin = lambda fam, i: fam in ("F1", "F2") or i % 3 == 0
    pb = heff.problem_from_workload(wlmod.lattice_workload("hubbard", 2, 14, seed=4, keep=thin))
    check_energy(pb, m_max=4)        # collapse restarts exercised


def test_steps_follow_the_oracle_iteration():
    """θ and ‖r‖ of every step against oracle/davidson.py on the same H_eff, diag and x0."""
    pb = heff.problem_from_workload(wlmod.lattice_workload("spinless", 6, 40, seed=5))
    H = heff.dense_heff(pb)
    dg = heff.psi_to_vec(pb, heff.diagonal_blockwise(pb))
    hist = []
    davidson.davidson(lambda v: H @ v, dg, heff.psi_to_vec(pb), tol=1e-9, m_max=6, history=hist)
    dp = device_problem(pb)
    dav = dp.davidson(m_max=6, tol=1e-9)
    dav.start(dp.psi_from_host(pb.psi))
    for i, (th_ref, rho_ref) in enumerate(hist):
        th, rho, conv = dav.step()
        assert abs(th - th_ref) <= 1e-9 * max(1.0, abs(th_ref)), i
        assert abs(rho - rho_ref) <= 1e-6 * max(rho_ref, 1e-3), i
        assert dav.query()[1] == min(i + 2, len(hist))      # exactly one apply per step
    assert conv


def test_config1_ground_energy():
    """BASELINE.json configs[0] hot call + Davidson: θ vs eigh of P†HP at the middle bond."""
    pb, Heff, _, _ = config1_problem()
    E = np.linalg.eigvalsh(Heff)[0]
    dp = device_problem(pb)
    dav = dp.davidson(m_max=16, tol=1e-9, max_iter=3000)
    dav.start(dp.psi_from_host(pb.psi))
    theta, rn, n_apply, ok = dav.solve(None)
    assert ok
    assert abs(theta - E) <= TOL_ENERGY * max(1.0, abs(E))


def test_not_converged_is_reported():
    pb = heff.problem_from_workload(wlmod.lattice_workload("spinless", 5, 24, seed=3))
    dp = device_problem(pb)
    dav = dp.davidson(m_max=4, tol=1e-13, max_iter=3)
    dav.start(dp.psi_from_host(pb.psi))
    theta, rn, n_apply, ok = dav.solve(None)
    assert not ok and n_apply == 3 and rn > 1e-13
