"""The CUDA path pinned to the mathematics directly (not through the oracle's solver): on a 4^4 lattice the
TSM estimator of Eq. 2.4, run end to end on the GPU (noise, HP and crude LP solves, contractions,
accumulation), must reproduce the exact traces sum_{x in t} tr[Gamma M^-1(x,x)] of the DENSE inverse within the
O(1/sqrt(N)) law of Eq. 2.1-2.3, whose variance for Z4 noise is known in closed form (pin P8).  The same for the
one-end estimators of Eq. 2.5 / 2.6 against the dense flavour difference / sum."""
import numpy as np
import pytest

import oracle
from dense_helpers import dense_from_apply, timeslice_projector_trace, volume
from paper_1211_0126_b200 import workloads as W

pytestmark = pytest.mark.gpu


def test_tsm_estimator_converges_to_the_dense_trace():
    from paper_1211_0126_b200 import tsm
    dims, kappa, mu, theta = (4, 4, 4, 4), 0.125, 0.25, -1
    U = W.random_su3_links(dims, 0.7, 404)
    V = volume(dims)
    M = dense_from_apply(lambda v: oracle.apply_M(dims, theta, kappa, mu, U, v), V)
    Md = dense_from_apply(lambda v: oracle.apply_M(dims, theta, kappa, -mu, U, v), V)
    Minv, Mdinv = np.linalg.inv(M), np.linalg.inv(Md)
    Lt, Vs = dims[3], V // dims[3]

    t = tsm.Tsm(dims, t_boundary=theta, max_nrhs=8)
    t.set_params(kappa, mu)
    t.set_gauge(U, 18)
    n_hp, n_lp = 16, 640
    got, secs, rc = t.run_loop_set(20121101, n_hp, n_lp, tsm.F32, 0.0, 2, hp_tol=1e-10, hp_max_iter=2000, nrhs=8,
                                   one_end=True, gen_one_end=True)
    assert rc == 0 and got.shape == (48, Lt)

    def variance(G, t_idx):   # Var[eta^dag A eta] = sum_{a != b} |A_ab|^2 for Z4 noise, A = P_t Gamma M^-1
        rows = slice(12 * Vs * t_idx, 12 * Vs * (t_idx + 1))
        A = np.kron(np.eye(Vs), np.kron(oracle.gamma(G), np.eye(3))) @ Minv[rows, :]
        tot = (np.abs(A) ** 2).sum()
        diag = (np.abs(np.diagonal(A[:, rows])) ** 2).sum()
        return tot - diag

    for G in (0, 1, 5):
        exact = timeslice_projector_trace(dims, oracle.gamma(G), Minv)
        for ti in range(Lt):
            sigma = np.sqrt(variance(G, ti) * (1.0 / n_lp + 1.0 / n_hp))
            assert abs(got[G, ti] - exact[ti]) < 6 * sigma, (G, ti, got[G, ti], exact[ti], sigma)
    # the scalar loop is large (a real signal many sigma above zero), so the check above is not vacuous
    exact0 = timeslice_projector_trace(dims, oracle.gamma(0), Minv)
    assert np.all(np.abs(exact0) > 50 * np.sqrt(variance(0, 0) / n_lp))

    # one-end trick (Eq. 2.5): tr[g5 (M_u^-1 - M_d^-1)]; generalised (Eq. 2.6): tr[1 (M_u^-1 + M_d^-1)]
    ex_diff = timeslice_projector_trace(dims, oracle.gamma(1), Minv - Mdinv)
    ex_sum = timeslice_projector_trace(dims, oracle.gamma(0), Minv + Mdinv)
    oe, goe = got[16 + 1], got[32 + 0]
    assert np.abs(oe - ex_diff).max() < 0.05 * np.abs(ex_diff).max()
    assert np.abs(goe - ex_sum).max() < 0.05 * np.abs(ex_sum).max()
    t.close()
