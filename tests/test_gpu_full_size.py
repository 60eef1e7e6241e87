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

  configs 2-5, loop level (north_star: "GPU loops match the oracle on all five workloads"):
      config 2 (8^3 x 16): the WHOLE Eq. 2.4 set (N_HP = 4, N_LP = 16) against the oracle, source by source;
      configs 3, 4, 5: the first HP and LP sources of the workload: per-source loops (all Gamma, all t; derivative
      loops at config 5) of the HP solve against the oracle's own HP solve (1e-8, A16(iii)), of the LP solve
      against the oracle's iterate at equal iteration count (fp32: 1e-4; bf16 storage: 2e-2), the (HP - LP)
      correction term of Eq. 2.4, the fp64 HP solve by oracle.true_residual, and the fp32 / 12-real stencil on
      the whole 16^3 x 32 lattice.

Tolerances as in test_gpu_parity.py; every one used here is listed in DESIGN.md section 7."""
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


def lp_args(wl):
    return {"f64": F64, "f32": F32, "bf16": BF16}[wl.lp_prec], wl.lp_tol, wl.lp_iters


def oracle_hp_lp(c, sid, k_lp):
    """The oracle's own HP solve (tol 1e-10) and its iterate after exactly k_lp iterations for source sid."""
    wl = c.wl
    eta = oracle.noise(wl.dims, wl.noise_seed, sid)
    s_hp, info_hp = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, wl.hp_tol, 5000)
    s_lp, _ = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, 0.0, k_lp)
    return eta, s_hp, info_hp, s_lp


def test_full_size_hp_loops_and_lp_at_the_workload_truncation_cfg5(cfg5):
    """Config 5 as the workload runs it: a 12-source fp64 HP batch (tol 1e-10) and the 12-source fp32 LP batch of
    the same sources at exactly 100 iterations, local + derivative loops.
      source 0: loops of the HP solve against the oracle's own HP solve, 1e-8 (A16(iii));
      source 1: the oracle certifies the GPU's s (fp64 true residual <= 1.5e-10, which bounds |s - M^-1 eta| by
                cond * 1e-10) and contracts that same s: 1e-12 (a second HP source without a second 150 s solve);
      LP, source 0: 100 iterations is past convergence (HP stops after ~53, reading A13), so the fp64 iterate
                after 100 iterations equals the HP solution to < 1e-10: the LP loops are compared with the
                oracle's HP loops at the fp32 bar 1e-4, and the (HP - LP) correction term of Eq. 2.4, which here
                measures fp32 rounding only, must stay below 1e-4 of the loops (the oracle's is < 1e-9)."""
    c, wl = cfg5, cfg5.wl
    ids = list(range(12))
    rc, info = c.t.solve(wl.noise_seed, ids, F64, wl.hp_tol, 5000, slot=0, want_true_resid=True)
    assert rc == 0 and all(i["rel_resid_true"] <= 1.5e-10 for i in info)
    rc, info_lp = c.t.solve(wl.noise_seed, ids, F32, 0.0, wl.lp_iters, slot=1)
    assert rc == 0 and all(i["iters"] == wl.lp_iters for i in info_lp)
    c.t.loops_reset(True)
    eta = oracle.noise(wl.dims, wl.noise_seed, 0)
    s_hp, info_hp = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, wl.hp_tol, 5000)
    assert abs(info[0]["iters"] - info_hp["iters"]) <= 1
    want_hp = oracle.all_loops(wl.dims, wl.t_boundary, c.U, eta, s_hp, True)
    got_hp, got_lp = c.t.loops_source(0, 0), c.t.loops_source(1, 0)
    assert got_hp.shape == want_hp.shape == (80, wl.dims[3])
    assert rel(c.t.get_solution(0, 0), s_hp) < 1e-9
    for lo, hi in ((0, 16), (16, 80)):
        assert rel(got_hp[lo:hi], want_hp[lo:hi]) < 1e-8, (lo, hi)
        assert rel(got_lp[lo:hi], want_hp[lo:hi]) < 1e-4, (lo, hi)
        assert np.abs(got_hp[lo:hi] - got_lp[lo:hi]).max() < 1e-4 * np.abs(want_hp[lo:hi]).max()
    # Eq. 2.4's correction term as the library accumulates it
    c.t.loops_add_correction(0, 1)
    corr, lp, n_hp, n_lp = c.t.loops_get_state()
    assert (n_hp, n_lp) == (12, 0) and not lp.any()
    sum_gpu = sum(c.t.loops_source(0, j) - c.t.loops_source(1, j) for j in range(12))
    assert np.abs(corr - sum_gpu).max() <= 1e-12 * np.abs(want_hp).max()
    # second HP source: certified by the oracle's residual, contracted by the oracle
    eta1 = oracle.noise(wl.dims, wl.noise_seed, 1)
    s1 = c.t.get_solution(0, 1)
    rho = oracle.true_residual(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta1, s1)
    assert rho <= 1.5e-10 and np.isclose(info[1]["rel_resid_true"], rho, rtol=1e-2)
    assert rel(c.t.loops_source(0, 1), oracle.all_loops(wl.dims, wl.t_boundary, c.U, eta1, s1, True)) < 1e-12
    c.t.loops_reset(True)


def test_full_eq_2_4_set_cfg2():
    """Config 2 in full (8^3 x 16, fp32 LP at 1e-3, fp64 HP at 1e-10, N_HP = 4, N_LP = 16, one source per batch):
    every per-source loop against the oracle -- HP at 1e-8, LP at equal iteration count at 1e-4 -- and the
    assembled Eq. 2.4 estimate against the same combination of the oracle's per-source loops."""
    c = Full(2, 1)
    wl = c.wl
    prec, tol, cap = lp_args(wl)
    got, secs, rc = c.t.run_loop_set(wl.noise_seed, wl.n_hp, wl.n_lp, prec, tol, cap, hp_tol=wl.hp_tol, hp_max_iter=5000, nrhs=wl.nrhs)
    assert rc == 0 and secs > 0
    per = {}
    want_tol = oracle.tsm_loops(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, wl.noise_seed, wl.n_hp, wl.n_lp,
                                wl.hp_tol, 5000, tol, cap, per_source=per)
    c.t.loops_reset(False)
    corr = np.zeros((16, wl.dims[3]), dtype=np.complex128)
    lp_sum = np.zeros_like(corr)
    same_iters = True
    for j in range(wl.n_hp + wl.n_lp):
        rc, info = c.t.solve(wl.noise_seed, [j], prec, tol, cap, slot=1, want_true_resid=True)
        assert rc == 0
        k = info[0]["iters"]
        assert abs(k - per[j]["info_lp"]["iters"]) <= 1 and info[0]["rel_resid_true"] <= 2 * tol      # A17
        same_iters &= k == per[j]["info_lp"]["iters"]
        eta = oracle.noise(wl.dims, wl.noise_seed, j)
        s_k, _ = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, 0.0, k)
        l_lp = oracle.loops(wl.dims, eta, s_k)
        got_lp = c.t.loops_source(1, 0)
        assert rel(got_lp, l_lp) < 1e-4, j
        if j < wl.n_hp:
            rc, info_hp = c.t.solve(wl.noise_seed, [j], F64, wl.hp_tol, 5000, slot=0)
            assert rc == 0 and abs(info_hp[0]["iters"] - per[j]["info_hp"]["iters"]) <= 1
            got_hp = c.t.loops_source(0, 0)
            assert rel(got_hp, per[j]["hp"]) < 1e-8, j
            # the (HP - LP) correction term, relative to its own size (it is O(tol) of the loops here)
            assert rel(got_hp - got_lp, per[j]["hp"] - l_lp) < 1e-3, j
            corr += per[j]["hp"] - l_lp
        else:
            lp_sum += l_lp
    want = corr / wl.n_hp + lp_sum / wl.n_lp
    assert rel(got, want) < 1e-4
    if same_iters:      # every fp32 solve stopped where the oracle's fp64 solve did: the oracle's own Eq. 2.4
        assert rel(got, want_tol) < 1e-4
    c.t.close()


def test_full_size_loops_cfg3_fp32_recon12():
    """Config 3 (16^3 x 32, 12-real links, single sources, LP = exactly 50 fp32 iterations): the fp32 / 12-real
    stencil on the whole lattice, and the first two HP sources (ids 0, 1) and LP-only sources (ids 8, 9)."""
    c = Full(3, 1)
    wl = c.wl
    assert c.dev < 1e-13
    psi = W.random_spinor(wl.dims, 3003, nrhs=1).astype(np.complex64).astype(np.complex128)
    want = oracle.hop(wl.dims, wl.t_boundary, c.U, psi[0] * c.odd[:, None, None], 0)
    assert rel(c.d_eo(F32, psi)[0], want) < 1e-5
    c.t.loops_reset(False)
    for sid in (0, 1, wl.n_hp, wl.n_hp + 1):
        hp = sid < wl.n_hp
        eta = oracle.noise(wl.dims, wl.noise_seed, sid)
        rc, info = c.t.solve(wl.noise_seed, [sid], F32, 0.0, wl.lp_iters, slot=1)
        assert rc == 0 and info[0]["iters"] == wl.lp_iters
        s_lp, _ = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, 0.0, wl.lp_iters)
        want_lp = oracle.loops(wl.dims, eta, s_lp)
        got_lp = c.t.loops_source(1, 0)
        assert rel(got_lp, want_lp) < 1e-4, sid
        if hp:
            rc, info = c.t.solve(wl.noise_seed, [sid], F64, wl.hp_tol, 5000, slot=0, want_true_resid=True)
            assert rc == 0 and info[0]["rel_resid_true"] <= 1.5e-10
            s_hp, info_hp = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, wl.hp_tol, 5000)
            assert abs(info[0]["iters"] - info_hp["iters"]) <= 1
            want_hp = oracle.loops(wl.dims, eta, s_hp)
            got_hp = c.t.loops_source(0, 0)
            assert rel(got_hp, want_hp) < 1e-8, sid
            # 50 iterations are past convergence (A13): the correction is fp32 rounding, the oracle's is < 1e-9
            assert np.abs(got_hp - got_lp).max() < 1e-4 * np.abs(want_hp).max()
            assert np.abs(want_hp - want_lp).max() < 1e-8 * np.abs(want_hp).max()
            if sid == 0:   # a truncation at which Eq. 2.4's correction term is sizeable: 5 iterations
                c.t.solve(wl.noise_seed, [sid], F32, 0.0, 5, slot=1)
                s5, _ = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, 0.0, 5)
                assert rel(got_hp - c.t.loops_source(1, 0), want_hp - oracle.loops(wl.dims, eta, s5)) < 1e-4
    c.t.close()


def test_full_size_loops_cfg4_bf16_batches():
    """Config 4 (24^3 x 48, bf16-storage LP at 5e-3, 12-real links, 4 sources per batch): HP sources 0, 1 and
    LP-only sources 16, 17 in one 4-source LP batch (a source's result does not depend on its batch, A14)."""
    c = Full(4, 4)
    wl = c.wl
    ids = [0, 1, wl.n_hp, wl.n_hp + 1]
    rc, info_lp = c.t.solve(wl.noise_seed, ids, BF16, wl.lp_tol, wl.lp_iters, slot=1, want_true_resid=True)
    assert rc == 0 and all(i["rel_resid_true"] <= 2 * wl.lp_tol for i in info_lp)
    rc, info_hp = c.t.solve(wl.noise_seed, ids[:2], F64, wl.hp_tol, 5000, slot=0, want_true_resid=True)
    assert rc == 0 and all(i["rel_resid_true"] <= 1.5e-10 for i in info_hp)
    c.t.loops_reset(False)
    got_lp = [c.t.loops_source(1, j) for j in range(4)]
    got_hp = [c.t.loops_source(0, j) for j in range(2)]
    for j, sid in enumerate(ids):
        eta = oracle.noise(wl.dims, wl.noise_seed, sid)
        k = info_lp[j]["iters"]
        s_k, _ = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, 0.0, k)
        want_lp = oracle.loops(wl.dims, eta, s_k)
        # bf16 storage of p, t, w (A20): the iterate carries 2^-8-sized relative perturbations
        assert rel(got_lp[j], want_lp) < 2e-2, sid
        if j == 0:
            s_hp, ref = oracle.solve(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, wl.hp_tol, 5000)
            assert abs(info_hp[0]["iters"] - ref["iters"]) <= 1
            want_hp = oracle.loops(wl.dims, eta, s_hp)
            assert rel(got_hp[0], want_hp) < 1e-8
            # Eq. 2.4's correction term is O(5e-3) of the loops here; bf16 perturbs it at the 2^-8 level of the LP part
            assert np.abs((got_hp[0] - got_lp[0]) - (want_hp - want_lp)).max() < 2e-2 * np.abs(want_lp).max()
        if j == 1:         # second HP source: certified by the oracle's residual, contracted by the oracle
            s1 = c.t.get_solution(0, 1)
            rho = oracle.true_residual(wl.dims, wl.t_boundary, wl.kappa, wl.mu, c.U, eta, s1)
            assert rho <= 1.5e-10
            assert rel(got_hp[1], oracle.loops(wl.dims, eta, s1)) < 1e-12
    c.t.close()


def test_full_size_cfg4_bf16_batch_of_4():
    c = Full(4, 4)
    wl = c.wl
    psi = W.random_spinor(wl.dims, 4004, nrhs=4)
    rounded = c.t.unpack(BF16, 4, c.t.pack(BF16, psi))
    got = c.d_eo(BF16, psi)
    for j in (0, 3):
        want = oracle.hop(wl.dims, wl.t_boundary, c.U, rounded[j] * c.odd[:, None, None], 0)
        assert rel_l2(got[j], want) < 1e-2                              # A20
        assert rel(got[j], want) < 1.5e-2                               # element by element
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
