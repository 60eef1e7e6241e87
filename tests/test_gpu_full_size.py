"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (same lattice,
precision, link storage and sources per batch), on outputs the oracle can afford:

  config 5 (32^3 x 64, fp32, 18-real links, 12 sources per batch, derivative loops): the stencil on the
      whole lattice for sampled sources of the batch, element by element; one truncated fp32 solve of a
      12-source batch against the oracle's iterate at equal iteration count and by fp64 true residual;
      the 80 per-timeslice loops of that source plus its one-end, generalised one-end and momentum-projected loops;
      a 12-source mixed-precision HP batch by fp64 true residual;
  config 4 (24^3 x 48, bf16 storage, 12-real links, 4 sources per batch): the stencil, and the solve at
      its residual truncation 5e-3 by true residual;
  config 3 (16^3 x 32, fp32, 12-real links, single source): 50 fixed iterations, true residual.

Tolerances as in test_gpu_parity.py."""
import numpy as np
import pytest

import oracle
from paper_1211_0126_b200 import workloads as W

pytestmark = pytest.mark.gpu

F64, F32, BF16 = 0, 1, 2


def rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def rel_l2(a, b):
    return np.linalg.norm((a - b).reshape(-1)) / np.linalg.norm(b.reshape(-1))


def parity_mask(dims):
    par = np.zeros(dims[::-1], dtype=np.int64)
    for ax in range(4):
        shape = [1, 1, 1, 1]
        shape[ax] = dims[::-1][ax]
        par = par + np.arange(dims[::-1][ax]).reshape(shape)
    return (par.reshape(-1) & 1)


class Full:
    def __init__(self, cfg, max_nrhs):
        from paper_1211_0126_b200 import tsm
        self.tsm = tsm
        self.wl = W.WORKLOADS[cfg]
        self.U = self.wl.links()
        self.t = tsm.Tsm(self.wl.dims, t_boundary=self.wl.t_boundary, max_nrhs=max_nrhs)
        self.t.set_params(self.wl.kappa, self.wl.mu)
        self.dev = self.t.set_gauge(self.U, self.wl.reconstruct)
        self.odd = parity_mask(self.wl.dims).astype(bool)

    def d_eo(self, prec, psi):
        """psi [nrhs][V][4][3] -> D_eo applied to its odd part, [nrhs][V][4][3] (odd sites zero)."""
        t, nrhs = self.t, psi.shape[0]
        fb = t.field_bytes(prec, nrhs)
        full_in = t.pack(prec, psi)
        full_out = t.alloc_field(prec, nrhs, full=True)
        t.dslash(self.tsm.OP_D_EO, prec, nrhs, full_in[fb:2 * fb], full_out[:fb])
        return t.unpack(prec, nrhs, full_out)


@pytest.fixture(scope="module")
def cfg5():
    f = Full(5, 12)
    yield f
    f.t.close()


def test_full_size_dslash_cfg5_fp32_batch_of_12(cfg5):
    c, wl = cfg5, cfg5.wl
    assert c.dev < 1e-13
    base = W.random_spinor(wl.dims, 5005, nrhs=3)
    psi = np.empty((12,) + base.shape[1:], dtype=np.complex128)
    for j in range(12):                                  # 12 distinct sources from 3 random fields
        psi[j] = (base[j % 3] * (1.0 + j // 3)).astype(np.complex64)
    del base
    got = c.d_eo(F32, psi)
    for j in (0, 7, 11):
        want = oracle.hop(wl.dims, wl.t_boundary, c.U, psi[j] * c.odd[:, None, None], 0)
        assert rel(got[j], want) < 1e-5, j
    # fp64, single source (the HP path's launch configuration)
    got64 = c.d_eo(F64, psi[:1])
    want = oracle.hop(wl.dims, wl.t_boundary, c.U, psi[0] * c.odd[:, None, None], 0)
    assert rel(got64[0], want) < 1e-12


def test_full_size_lp_solve_and_loops_cfg5(cfg5):
    c, wl = cfg5, cfg5.wl
    ids = list(range(40, 52))
    k = 4
    rc, info = c.t.solve(wl.noise_seed, ids, F32, 0.0, k, slot=1, want_true_resid=True)
    assert rc == 0 and all(i["iters"] == k for i in info)
    j = 5
    eta = oracle.noise(wl.dims, wl.noise_seed, ids[j])
    s_ref, info_ref = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, 0.0, k)
    s = c.t.get_solution(1, j)
    assert rel(s, s_ref) < 2e-5                                         # equal iteration count, early iterate
    rho = oracle.true_residual(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, s)
    assert rho <= max(2 * info_ref["rel_resid_true"], 100 * 6e-8)       # A17, fixed-k mode
    assert np.isclose(info[j]["rel_resid_true"], rho, rtol=1e-3)
    moms = [(1, 0, 0), (0, -1, 1)]
    c.t.loops_reset(True, one_end=True, gen_one_end=True, momenta=moms)
    got = c.t.loops_source(1, j)
    want = oracle.all_loops(wl.dims, wl.t_boundary, c.U, eta, s_ref, True, one_end=(wl.kappa, wl.mu),
                            gen_one_end=wl.kappa, momenta=moms)             # the oracle's own iterate
    assert got.shape == want.shape == (80 + 16 + 16 + 32, wl.dims[3])
    for lo, hi in ((0, 16), (16, 80), (80, 96), (96, 112), (112, 144)):      # s agrees to 2e-5 elementwise
        assert rel(got[lo:hi], want[lo:hi]) < 1e-4, (lo, hi)
    c.t.loops_reset(True)


def test_full_size_mixed_precision_hp_batch_cfg5(cfg5):
    """N4 at the headline size: 12 sources, fp64 defect correction around the fp32 CG to 1e-10; the oracle checks
    the fp64 true residual of the full system for a sampled source."""
    c, wl = cfg5, cfg5.wl
    rc, info = c.t.solve(wl.noise_seed, list(range(12)), c.tsm.MIXED, wl.hp_tol, 5000, slot=0, want_true_resid=True)
    assert rc == 0
    assert all(i["status"] == 0 and i["rel_resid_rec"] <= wl.hp_tol and i["rel_resid_true"] <= 1.5e-10 for i in info)
    eta = oracle.noise(wl.dims, wl.noise_seed, 7)
    rho = oracle.true_residual(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, c.t.get_solution(0, 7))
    assert rho <= 1.5e-10 and np.isclose(info[7]["rel_resid_true"], rho, rtol=1e-2)


def test_full_size_cfg5_100_iterations_reach_the_fp32_floor(cfg5):
    """The headline launch configuration itself: 12 sources, exactly 100 fp32 iterations (past convergence,
    reading A13): every source reports 100 iterations, no breakdown, and an fp64 true residual at the fp32 floor."""
    c, wl = cfg5, cfg5.wl
    rc, info = c.t.solve(wl.noise_seed, list(range(12)), F32, 0.0, wl.lp_iters, slot=1, want_true_resid=True)
    assert rc == 0
    for i in info:
        assert i["iters"] == wl.lp_iters and i["status"] == 0
        assert i["rel_resid_true"] < 100 * 6e-8
    eta = oracle.noise(wl.dims, wl.noise_seed, 3)
    rho = oracle.true_residual(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, c.t.get_solution(1, 3))
    assert np.isclose(info[3]["rel_resid_true"], rho, rtol=1e-2)


def test_full_size_cfg4_bf16_batch_of_4():
    c = Full(4, 4)
    wl = c.wl
    psi = W.random_spinor(wl.dims, 4004, nrhs=4)
    rounded = c.t.unpack(BF16, 4, c.t.pack(BF16, psi))
    got = c.d_eo(BF16, psi)
    for j in (0, 3):
        want = oracle.hop(wl.dims, wl.t_boundary, c.U, rounded[j] * c.odd[:, None, None], 0)
        assert rel_l2(got[j], want) < 1e-2                              # A20
    ids = [0, 1, 2, 3]
    rc, info = c.t.solve(wl.noise_seed, ids, BF16, wl.lp_tol, wl.lp_iters, slot=1, want_true_resid=True)
    assert rc == 0
    j = 2
    eta = oracle.noise(wl.dims, wl.noise_seed, ids[j])
    _, info_ref = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, wl.lp_tol, wl.lp_iters)
    assert abs(info[j]["iters"] - info_ref["iters"]) <= 2
    rho = oracle.true_residual(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, c.t.get_solution(1, j))
    assert rho <= 2 * wl.lp_tol
    assert all(i["rel_resid_true"] <= 2 * wl.lp_tol for i in info)
    c.t.close()


def test_full_size_cfg3_fp32_recon12_50_iterations():
    c = Full(3, 1)
    wl = c.wl
    rc, info = c.t.solve(wl.noise_seed, [9], F32, 0.0, wl.lp_iters, slot=1, want_true_resid=True)
    assert rc == 0 and info[0]["iters"] == wl.lp_iters
    eta = oracle.noise(wl.dims, wl.noise_seed, 9)
    _, info_ref = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, 0.0, wl.lp_iters)
    rho = oracle.true_residual(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, c.t.get_solution(1, 0))
    assert rho <= max(2 * info_ref["rel_resid_true"], 100 * 6e-8)
    c.t.close()
