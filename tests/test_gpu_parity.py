"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element on
the same seeded inputs.  Tolerances: bit-exact noise and
indexing; 1e-12 relative for fp64 stencil and HP loops; 1e-5 for fp32 stencil; 1e-2 for
bf16 storage (A20); LP solves by true residual (A17)."""
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


@pytest.fixture(scope="module")
def tsm_mod():
    from paper_1211_0126_b200 import tsm
    return tsm


class Case:
    def __init__(self, tsm_mod, dims, eps, seed, kappa, mu, theta, max_nrhs=4, recon=18):
        self.dims, self.kappa, self.mu, self.theta = dims, kappa, mu, theta
        self.U = W.random_su3_links(dims, eps, seed)
        self.t = tsm_mod.Tsm(dims, t_boundary=theta, max_nrhs=max_nrhs)
        self.t.set_params(kappa, mu)
        self.dev = self.t.set_gauge(self.U, recon)
        par = np.zeros(dims[::-1], dtype=np.int64)
        for ax in range(4):
            shape = [1, 1, 1, 1]
            shape[ax] = dims[::-1][ax]
            par = par + np.arange(dims[::-1][ax]).reshape(shape)
        self.par = (par.reshape(-1) & 1)


@pytest.fixture(scope="module")
def small(tsm_mod):
    wl = W.WORKLOADS[1]
    return Case(tsm_mod, wl.dims, wl.eps, wl.gauge_seed, wl.kappa, wl.mu, -1, max_nrhs=4)


@pytest.fixture(scope="module")
def ragged(tsm_mod):
    # extents that are not multiples of anything convenient: V_h = 6*10*4*6/2 = 720 sites
    return Case(tsm_mod, (6, 10, 4, 6), 0.6, 77, 0.157, 0.02, +1, max_nrhs=12)


@pytest.fixture(scope="module")
def medium(tsm_mod):
    wl = W.WORKLOADS[2]
    return Case(tsm_mod, wl.dims, wl.eps, wl.gauge_seed, wl.kappa, wl.mu, -1, max_nrhs=4)


# ---------------------------------------------------------------- H1/H3: indexing and noise, bit-exact
@pytest.mark.parametrize("kind", [0, 1])
def test_noise_bit_exact(small, ragged, kind):
    for c in (small, ragged):
        for sid in (0, 5, 4000000000):
            seed = 0x1211012600000001
            got = c.t.noise(seed, sid, kind)
            want = oracle.noise(c.dims, seed, sid, kind)
            assert np.array_equal(got, want)


def test_pack_unpack_round_trip_is_exact(ragged):
    c = ragged
    psi = W.random_spinor(c.dims, 5, nrhs=3)
    buf = c.t.pack(F64, psi)
    assert np.array_equal(c.t.unpack(F64, 3, buf), psi)
    # fp32 / bf16 storage round the values once, nothing else
    assert np.array_equal(c.t.unpack(F32, 3, c.t.pack(F32, psi)), psi.astype(np.complex64).astype(np.complex128))
    b = c.t.unpack(BF16, 3, c.t.pack(BF16, psi))
    assert rel(b, psi) < 2 ** -8


def test_gauge_ingest_reports_unitarity(small, tsm_mod):
    assert small.dev < 1e-13
    bad = small.U.copy()
    bad[2, 17] *= 1.001
    t = tsm_mod.Tsm(small.dims, max_nrhs=1)
    assert abs(t.set_gauge(bad, 18) - 0.003) < 1e-3       # accepted with 18 reals, deviation reported
    with pytest.raises(tsm_mod.TsmError) as e:
        t.set_gauge(bad, 12)
    assert e.value.code == tsm_mod.ENOTUNITARY
    t.close()


# ---------------------------------------------------------------- H5: the stencil
def _oracle_op(c, op, psi):
    """psi: full-lattice [V][4][3]; returns the full-lattice oracle result of operator `op`."""
    e = (c.par == 0)[:, None, None]
    if op == 0:
        return oracle.hop(c.dims, c.theta, c.U, psi * ~e, 0)
    if op == 1:
        return oracle.hop(c.dims, c.theta, c.U, psi * e, 1)
    if op == 2:
        return oracle.apply_Mhat(c.dims, c.theta, c.kappa, c.mu, c.U, psi * e)
    if op == 3:
        return oracle.apply_Mhat_dag(c.dims, c.theta, c.kappa, c.mu, c.U, psi * e)
    return oracle.apply_M(c.dims, c.theta, c.kappa, c.mu, c.U, psi)


def _gpu_op(c, op, prec, psi):
    """psi: [nrhs][V][4][3].  Packs, applies, unpacks; unused parities come back as zeros."""
    nrhs = psi.shape[0]
    t = c.t
    fb = t.field_bytes(prec, nrhs)
    full_in = t.pack(prec, psi)
    full_out = t.alloc_field(prec, nrhs, full=True)
    if op == 4:
        t.dslash(op, prec, nrhs, full_in, full_out)
    else:
        in_par = {0: 1, 1: 0, 2: 0, 3: 0}[op]
        out_par = {0: 0, 1: 1, 2: 0, 3: 0}[op]
        t.dslash(op, prec, nrhs, full_in[in_par * fb:(in_par + 1) * fb], full_out[out_par * fb:(out_par + 1) * fb])
    return t.unpack(prec, nrhs, full_out)


@pytest.mark.parametrize("op", [0, 1, 2, 3, 4])
def test_dslash_fp64_parity(small, ragged, medium, op):
    for c in (small, ragged, medium):
        psi = W.random_spinor(c.dims, 100 + op, nrhs=1)
        got = _gpu_op(c, op, F64, psi)[0]
        want = _oracle_op(c, op, psi[0])
        assert rel(got, want) < 1e-12, (c.dims, op)


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("op", [0, 1, 2, 3, 4])
def test_dslash_fp32_parity(tsm_mod, op, recon):
    for dims, theta in [((4, 4, 4, 8), -1), ((6, 10, 4, 6), +1)]:
        c = Case(tsm_mod, dims, 0.6, 81, 0.157, 0.02, theta, max_nrhs=2, recon=recon)
        psi = W.random_spinor(dims, 200 + op, nrhs=1)
        got = _gpu_op(c, op, F32, psi)[0]
        # the oracle sees the same fp32-rounded input (links stay fp64 on its side)
        want = _oracle_op(c, op, psi[0].astype(np.complex64).astype(np.complex128))
        assert rel(got, want) < 1e-5, (dims, op, recon)
        c.t.close()


@pytest.mark.parametrize("op", [0, 3, 4])
def test_dslash_bf16_storage_parity(ragged, op):
    c = ragged
    psi = W.random_spinor(c.dims, 300 + op, nrhs=1)
    rounded = c.t.unpack(BF16, 1, c.t.pack(BF16, psi))
    got = _gpu_op(c, op, BF16, psi)[0]
    want = _oracle_op(c, op, rounded[0])
    assert rel_l2(got, want) < 1e-2
    # element by element: every stored value is one bf16 rounding (2^-9 relative) of an
    # fp32 result whose intermediates (the t field of Mhat) were bf16 as well
    assert rel(got, want) < 1.5e-2


@pytest.mark.parametrize("nrhs", [2, 3, 4, 12])
@pytest.mark.parametrize("prec,tol", [(F64, 1e-12), (F32, 1e-5)])
def test_dslash_multi_rhs(ragged, nrhs, prec, tol):
    c = ragged
    psi = W.random_spinor(c.dims, 400 + nrhs, nrhs=nrhs)
    for op in (0, 2, 4):
        got = _gpu_op(c, op, prec, psi)
        for j in range(nrhs):
            src = psi[j] if prec == F64 else psi[j].astype(np.complex64).astype(np.complex128)
            assert rel(got[j], _oracle_op(c, op, src)) < tol, (op, j)


# ---------------------------------------------------------------- H4/H6/H7: solves
def test_hp_solve_matches_oracle(small, medium, tsm_mod):
    for c, seed in ((small, W.WORKLOADS[1].noise_seed), (medium, W.WORKLOADS[2].noise_seed)):
        eta = oracle.noise(c.dims, seed, 1)
        s_ref, info_ref = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 1e-10, 2000)
        rc, info = c.t.solve(seed, [1], F64, 1e-10, 2000, slot=0, want_true_resid=True)
        assert rc == 0 and info[0]["status"] == 0
        assert info[0]["iters"] == info_ref["iters"]
        assert np.isclose(info[0]["rel_resid_rec"], info_ref["rel_resid_rec"], rtol=1e-6)
        s = c.t.get_solution(0, 0)
        rho = oracle.true_residual(c.dims, c.theta, c.kappa, c.mu, c.U, eta, s)
        assert rho <= 1.5e-10                                              # A16(iii)
        assert np.isclose(info[0]["rel_resid_true"], rho, rtol=1e-3)
        assert rel(s, s_ref) < 1e-11
        # same fixed iteration count: identical recurrences, rounding-order differences only (A16(ii))
        k = info_ref["iters"]
        s_fix_ref, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 0.0, k)
        rc, info = c.t.solve(seed, [1], F64, 0.0, k, slot=1)
        assert rc == 0 and info[0]["iters"] == k
        assert rel(c.t.get_solution(1, 0), s_fix_ref) < 1e-12


def test_truncated_solves_match_oracle_iterates(small):
    """fp64 LP (config 1): same recurrences, so the truncated iterate itself matches."""
    c = small
    seed = W.WORKLOADS[1].noise_seed
    eta = oracle.noise(c.dims, seed, 3)
    for tol, k in ((1e-2, 1000), (0.0, 1), (0.0, 2), (0.0, 5)):
        s_ref, info_ref = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, tol, k)
        rc, info = c.t.solve(seed, [3], F64, tol, k, slot=0)
        assert rc == 0
        assert info[0]["iters"] == info_ref["iters"]
        assert rel(c.t.get_solution(0, 0), s_ref) < 1e-12
    # tolerance not reached: flagged, iterate kept (8(b))
    rc, info = c.t.solve(seed, [3], F64, 1e-12, 3, slot=0)
    assert rc == -6 and info[0]["status"] == -6 and info[0]["iters"] == 3
    s_ref, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 0.0, 3)
    assert rel(c.t.get_solution(0, 0), s_ref) < 1e-12


def test_fp32_lp_solves_by_true_residual(medium):
    """A17: residual mode rho <= 2 tol and |iters - oracle| <= 1; fixed-k mode rho <= max(2 rho_oracle, 100 eps)."""
    c = medium
    wl = W.WORKLOADS[2]
    for sid in (0, 7):
        eta = oracle.noise(c.dims, wl.noise_seed, sid)
        _, info_ref = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, wl.lp_tol, 1000)
        rc, info = c.t.solve(wl.noise_seed, [sid], F32, wl.lp_tol, 1000, slot=1, want_true_resid=True)
        assert rc == 0
        assert abs(info[0]["iters"] - info_ref["iters"]) <= 1
        s = c.t.get_solution(1, 0)
        rho = oracle.true_residual(c.dims, c.theta, c.kappa, c.mu, c.U, eta, s)
        assert rho <= 2 * wl.lp_tol
        assert np.isclose(info[0]["rel_resid_true"], rho, rtol=1e-3)
        for k in (5, 20, 60):
            s_ref, info_ref = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 0.0, k)
            rc, info = c.t.solve(wl.noise_seed, [sid], F32, 0.0, k, slot=1)
            assert rc == 0 and info[0]["iters"] == k
            s = c.t.get_solution(1, 0)
            rho = oracle.true_residual(c.dims, c.theta, c.kappa, c.mu, c.U, eta, s)
            assert rho <= max(2 * info_ref["rel_resid_true"], 100 * 6e-8)
            if k == 5:   # equal iteration count, early iterate: elementwise to fp32 accuracy
                assert rel(s, s_ref) < 2e-5


def test_batched_solve_is_independent_of_batch_composition(medium):
    """A14: batched, not block, CG: each source gets the iterate it would get alone."""
    c = medium
    seed = W.WORKLOADS[2].noise_seed
    rc, info = c.t.solve(seed, [4, 9, 2, 11], F64, 1e-6, 500, slot=0)
    assert rc == 0
    batch = [c.t.get_solution(0, j) for j in range(4)]
    for j, sid in enumerate([4, 9, 2, 11]):
        rc, single = c.t.solve(seed, [sid], F64, 1e-6, 500, slot=1)
        assert single[0]["iters"] == info[j]["iters"]
        assert np.array_equal(c.t.get_solution(1, 0), batch[j])
    assert len({i["iters"] for i in info}) >= 1


# ---------------------------------------------------------------- H8/H9: contractions
@pytest.mark.parametrize("deriv", [False, True])
def test_contraction_parity_on_the_oracle_solution(small, ragged, deriv):
    """A16(i): feed the oracle's s to the GPU contraction; 1e-12 relative to the largest loop."""
    for c in (small, ragged):
        seed = 99
        c.t.loops_reset(deriv)
        rc, _ = c.t.solve(seed, [2, 6], F64, 0.0, 1, slot=0)     # registers the source ids of the slot
        for j, sid in enumerate((2, 6)):
            eta = oracle.noise(c.dims, seed, sid)
            s, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 1e-10, 2000)
            c.t.set_solution(0, j, s)
            want = oracle.all_loops(c.dims, c.theta, c.U, eta, s, deriv)
            got = c.t.loops_source(0, j)
            assert got.shape == want.shape
            assert rel(got, want) < 1e-12


def _oracle_solution_in_fp32_slot(c, seed, ids, k):
    """Registers `ids` in slot 1 (an fp32 solve), then overwrites the slot with the ORACLE's k-iteration solutions;
    returns them rounded to fp32 in numpy, which is what the slot now holds (no oracle input comes from the GPU)."""
    rc, _ = c.t.solve(seed, ids, F32, 0.0, 1, slot=1)
    out = []
    for j, sid in enumerate(ids):
        eta = oracle.noise(c.dims, seed, sid)
        s, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 0.0, k)
        c.t.set_solution(1, j, s)
        out.append((eta, s.astype(np.complex64).astype(np.complex128)))
    return out


def test_contraction_fp32_slot(ragged):
    c = ragged
    c.t.loops_reset(True)
    (eta, s32), = _oracle_solution_in_fp32_slot(c, 5, [1], 30)
    want = oracle.all_loops(c.dims, c.theta, c.U, eta, s32, True)
    got = c.t.loops_source(1, 0)
    # fp32 values; per lane the 4 x 4 spin matrices of up to 4 sites and the warp's 32 lanes are added in fp32 (the
    # transposed butterfly), everything beyond that in fp64: 1e-6 of the largest loop
    assert rel(got[:16], want[:16]) < 1e-6
    assert rel(got[16:], want[16:]) < 1e-5           # covariant difference in fp32 arithmetic


# ---------------------------------------------------------------- H10: Eq. 2.4
def test_tsm_loop_set_config1(small):
    """Config 1 in full: fp64 throughout, N_HP=2, N_LP=4, LP at 1e-2 (A11: 6 sources)."""
    c = small
    wl = W.WORKLOADS[1]
    c.t.set_hp_precision(F64)      # "fp64 throughout"; the library's default HP solver is the mixed-precision one
    per = {}
    want = oracle.tsm_loops(c.dims, c.theta, c.kappa, c.mu, c.U, wl.noise_seed, wl.n_hp, wl.n_lp,
                            wl.hp_tol, 2000, wl.lp_tol, wl.lp_iters, with_derivative=True, per_source=per)
    got, secs, rc = c.t.run_loop_set(wl.noise_seed, wl.n_hp, wl.n_lp, F64, wl.lp_tol, wl.lp_iters,
                                     hp_tol=wl.hp_tol, hp_max_iter=2000, nrhs=1, with_derivative=True)
    assert rc == 0 and secs > 0
    # HP solves stop at 1e-10, so HP loops agree to ~cond*tol (A16(iii)); LP iterates agree to rounding
    assert rel(got, want) < 1e-8
    # batching must not change anything: same set with 2 sources per batch
    got2, _, _ = c.t.run_loop_set(wl.noise_seed, wl.n_hp, wl.n_lp, F64, wl.lp_tol, wl.lp_iters,
                                  hp_tol=wl.hp_tol, hp_max_iter=2000, nrhs=2, with_derivative=True)
    assert np.array_equal(got, got2)
    # LP == HP: the correction vanishes identically and Eq. 2.4 is Eq. 2.2 over the LP set (P11)
    got3, _, _ = c.t.run_loop_set(wl.noise_seed, 2, 3, F64, 1e-9, 2000, hp_tol=1e-9, hp_max_iter=2000, nrhs=1)
    corr, lp, n_hp, n_lp = c.t.loops_get_state()
    assert n_hp == 2 and n_lp == 3 and not corr.any()
    assert np.array_equal(got3, lp / 3)
    # the default HP solver (fp64 defect correction around the fp32 CG) gives the same estimate to the HP tolerance
    c.t.set_hp_precision(3)
    got4, _, rc = c.t.run_loop_set(wl.noise_seed, wl.n_hp, wl.n_lp, F64, wl.lp_tol, wl.lp_iters,
                                   hp_tol=wl.hp_tol, hp_max_iter=2000, nrhs=1, with_derivative=True)
    assert rc == 0 and rel(got4, want) < 1e-8


def test_tsm_manual_accumulation_and_state(small):
    c = small
    seed = 31
    c.t.loops_reset(False)
    c.t.solve(seed, [0, 1], F64, 1e-10, 2000, slot=0)
    c.t.solve(seed, [0, 1], F64, 0.0, 3, slot=1)
    l_hp = [c.t.loops_source(0, j) for j in range(2)]
    l_lp = [c.t.loops_source(1, j) for j in range(2)]
    c.t.loops_add_correction(0, 1)
    c.t.solve(seed, [2, 3, 4], F64, 0.0, 3, slot=1)
    l_lp2 = [c.t.loops_source(1, j) for j in range(3)]
    c.t.loops_add_lp(1)
    got = c.t.loops_finalize()
    want = (l_hp[0] - l_lp[0] + l_hp[1] - l_lp[1]) / 2 + sum(l_lp2) / 3
    assert rel(got, want) < 1e-14
    corr, lp, n_hp, n_lp = c.t.loops_get_state()
    assert (n_hp, n_lp) == (2, 3)
    c.t.loops_reset(False)
    c.t.loops_set_state(corr, lp, n_hp, n_lp)           # resume
    assert np.array_equal(c.t.loops_finalize(), got)
    # Eq. 2.4 needs the same eta_j on both sides
    c.t.solve(seed, [5, 6, 7], F64, 0.0, 3, slot=0)
    c.t.solve(seed, [5, 6, 8], F64, 0.0, 3, slot=1)
    with pytest.raises(Exception):
        c.t.loops_add_correction(0, 1)


# ---------------------------------------------------------------- error behaviour (8(b))
def test_state_and_argument_errors(tsm_mod):
    t = tsm_mod.Tsm((4, 4, 4, 4), max_nrhs=2)
    with pytest.raises(tsm_mod.TsmError) as e:
        t.solve(1, [0], F64, 1e-6, 10)
    assert e.value.code == tsm_mod.ESTATE                # no gauge / params yet
    t.set_gauge(W.unit_links((4, 4, 4, 4)))
    with pytest.raises(tsm_mod.TsmError) as e:
        t.solve(1, [0], F64, 1e-6, 10)
    assert e.value.code == tsm_mod.ESTATE
    t.set_params(0.12, 0.1)
    with pytest.raises(tsm_mod.TsmError) as e:
        t.solve(1, [0, 1, 2], F64, 1e-6, 10)             # nrhs > max_nrhs
    assert e.value.code == tsm_mod.EINVAL
    with pytest.raises(tsm_mod.TsmError) as e:
        t.get_solution(1, 0)                             # empty slot
    assert e.value.code == tsm_mod.ESTATE
    rc, info = t.solve(1, [0], F64, 1e-8, 200)
    assert rc == 0
    with pytest.raises(tsm_mod.TsmError):
        tsm_mod.Tsm((4, 4, 5, 4))
    t.close()


def test_single_source_context_solution_round_trip(tsm_mod):
    """max_nrhs = 1 (the default of Tsm(), and what configs 1-3 use): get_solution / set_solution of an fp64 slot
    must not touch the other slot or the other parity (the gather buffer used to overlap slot 0)."""
    wl = W.WORKLOADS[1]
    U = wl.links()
    t = tsm_mod.Tsm(wl.dims, t_boundary=-1, max_nrhs=1)
    t.set_params(wl.kappa, wl.mu)
    t.set_gauge(U, 18)
    eta = oracle.noise(wl.dims, wl.noise_seed, 3)
    s_ref, info_ref = oracle.solve(wl.dims, -1, wl.kappa, wl.mu, U, eta, wl.hp_tol, 2000)
    rc, info = t.solve(wl.noise_seed, [3], F64, wl.hp_tol, 2000, slot=0)
    assert rc == 0 and info[0]["iters"] == info_ref["iters"]
    rc, _ = t.solve(wl.noise_seed, [3], F64, 0.0, 3, slot=1)
    s1 = t.get_solution(1, 0)
    s0 = t.get_solution(0, 0)
    assert rel(s0, s_ref) < 1e-11
    assert np.array_equal(t.get_solution(0, 0), s0) and np.array_equal(t.get_solution(1, 0), s1)   # reads change nothing
    assert rel(t.loops_source(0, 0), oracle.loops(wl.dims, eta, s_ref)) < 1e-8                       # slot 0 still whole
    assert rel(t.loops_source(0, 0), oracle.loops(wl.dims, eta, s0)) < 1e-12
    t.set_solution(0, 0, s_ref)
    assert np.array_equal(t.get_solution(0, 0), s_ref)                                                # both parities
    assert np.array_equal(t.get_solution(1, 0), s1)
    assert rel(t.loops_source(0, 0), oracle.loops(wl.dims, eta, s_ref)) < 1e-12
    t.close()


def test_non_finite_links_are_refused(tsm_mod):
    dims = (4, 4, 4, 4)
    t = tsm_mod.Tsm(dims, max_nrhs=1)
    for bad_value in (np.nan, np.inf):
        U = W.unit_links(dims)
        U[1, 5, 2, 2] = bad_value
        for recon in (18, 12):
            with pytest.raises(tsm_mod.TsmError) as e:
                t.set_gauge(U, recon)
            assert e.value.code == tsm_mod.EINVAL
    with pytest.raises(tsm_mod.TsmError) as e:
        t.set_params(0.1, 0.1)
        t.solve(1, [0], F64, 1e-6, 10)                   # the refused field is not usable
    assert e.value.code == tsm_mod.ESTATE
    t.close()


def test_loop_calls_need_a_reset_after_set_momenta(small, tsm_mod):
    import ctypes
    t = tsm_mod.Tsm(small.dims, max_nrhs=1)
    t.set_params(small.kappa, small.mu)
    t.set_gauge(small.U, 18)
    t.solve(7, [0], F64, 0.0, 2, slot=1)
    z = t.loops_finalize()                               # before any reset: the default 16 loops, zeroed sums
    assert z.shape == (16, small.dims[3]) and not z.any()
    mom = (ctypes.c_int * 3)(1, 0, 0)
    assert t.lib.tsm_loops_set_momenta(t._h, 1, mom) == 0
    out = np.empty((32, small.dims[3]), dtype=np.complex128)
    dp = out.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
    assert t.lib.tsm_loops_add_lp(t._h, 1) == tsm_mod.ESTATE
    assert t.lib.tsm_loops_finalize(t._h, dp) == tsm_mod.ESTATE
    assert t.lib.tsm_loops_source(t._h, 1, 0, dp) == tsm_mod.ESTATE
    t.loops_reset(momenta=[(1, 0, 0)])
    t.loops_add_lp(1)
    assert np.isfinite(t.loops_finalize().view(np.float64)).all()
    t.close()


# ---------------------------------------------------------------- bf16 storage (config 4) and fp32 batches
def test_bf16_lp_solves_by_true_residual(tsm_mod):
    """A17 for bf16 storage: config 4's parameters on an 8^3 x 16 lattice, 4 sources per batch, tol 5e-3:
    fp64 true residual of the full system <= 2 tol, iteration count within 2 of the oracle's."""
    wl = W.WORKLOADS[4]
    c = Case(tsm_mod, (8, 8, 8, 16), wl.eps, wl.gauge_seed, wl.kappa, wl.mu, -1, max_nrhs=4, recon=12)
    ids = [0, 1, 2, 3]
    rc, info = c.t.solve(wl.noise_seed, ids, BF16, wl.lp_tol, 1000, slot=1, want_true_resid=True)
    assert rc == 0
    for j, sid in enumerate(ids):
        eta = oracle.noise(c.dims, wl.noise_seed, sid)
        _, info_ref = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, wl.lp_tol, 1000)
        assert abs(info[j]["iters"] - info_ref["iters"]) <= 2, (info[j], info_ref)
        rho = oracle.true_residual(c.dims, c.theta, c.kappa, c.mu, c.U, eta, c.t.get_solution(1, j))
        assert rho <= 2 * wl.lp_tol, rho
        assert np.isclose(info[j]["rel_resid_true"], rho, rtol=1e-3)
    # fixed-k mode: rho <= max(2 rho_oracle(k), 100 eps_bf16) with eps_bf16 = 2^-8
    eta = oracle.noise(c.dims, wl.noise_seed, 0)
    for k in (3, 12):
        _, info_ref = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 0.0, k)
        rc, info = c.t.solve(wl.noise_seed, [0, 1], BF16, 0.0, k, slot=1)
        assert rc == 0 and info[0]["iters"] == k
        rho = oracle.true_residual(c.dims, c.theta, c.kappa, c.mu, c.U, eta, c.t.get_solution(1, 0))
        assert rho <= max(2 * info_ref["rel_resid_true"], 100 * 2.0 ** -8)
    c.t.close()


@pytest.mark.parametrize("prec", [F32, BF16])
def test_low_precision_batches_are_independent_of_batch_composition(medium, ragged, prec):
    """A14 in the LP precisions: the batched kernels (shared-memory link tiles, several sources per CTA)
    and the single-source kernel give a source the same iterate, bit for bit."""
    for c in (medium, ragged):
        seed = 4242
        ids = [4, 9, 2, 11, 7]
        rc, info = c.t.solve(seed, ids[:4], prec, 0.0, 6, slot=0)
        assert rc == 0
        batch = [c.t.get_solution(0, j) for j in range(4)]
        for j in (0, 3):
            rc, single = c.t.solve(seed, [ids[j]], prec, 0.0, 6, slot=1)
            assert np.array_equal(c.t.get_solution(1, 0), batch[j]), (c.dims, prec, j)
        rc, _ = c.t.solve(seed, [ids[3], ids[4], ids[0]], prec, 0.0, 6, slot=1)   # other batch, other position
        assert np.array_equal(c.t.get_solution(1, 0), batch[3])
        assert np.array_equal(c.t.get_solution(1, 2), batch[0])


def test_cuda_graph_chunks_equal_kernel_by_kernel_launches(medium):
    """Later chunks of 4 CG iterations run as one cached CUDA graph; with per-launch profiling on the same
    iterations are launched kernel by kernel.  Same kernels, same order: bit-identical iterates."""
    c = medium
    seed = 777
    for prec, tol, k in ((F64, 1e-10, 2000), (F32, 0.0, 23), (BF16, 0.0, 9)):
        c.t.profile(False)
        rc, info_g = c.t.solve(seed, [3, 8], prec, tol, k, slot=0)
        a = [c.t.get_solution(0, j) for j in range(2)]
        c.t.profile(True)
        rc, info_d = c.t.solve(seed, [3, 8], prec, tol, k, slot=1)
        c.t.profile(False)
        for kind in range(5):
            c.t.profile_read(prec, kind)
        assert [i["iters"] for i in info_g] == [i["iters"] for i in info_d]
        for j in range(2):
            assert np.array_equal(a[j], c.t.get_solution(1, j)), (prec, j)
    # the three launch modes (kernel by kernel, graphs of 4 iterations, device-side WHILE loop) give the same iterates
    # and the same launch count: noise, twist, 3 stencils, init; per iteration 4 stencils + update (k_dslash_small
    # finishes its own reductions on this lattice); the loop's begin kernel; reconstruction
    ref = None
    for mode in (0, 1, 1, 2, 2, 3, 4):
        c.t.set_graphs(mode)
        for tol, k in ((0.0, 12), (1e-4, 500)):
            n0 = c.t.launch_count()
            rc, info = c.t.solve(seed, [3, 5], F32, tol, k, slot=0)
            n_l = c.t.launch_count() - n0
            got = (info[0]["iters"], info[1]["iters"], c.t.get_solution(0, 0), c.t.get_solution(0, 1))
            if tol == 0.0:
                # 3: ONE launch for the loop; 4 (automatic, this lattice): noise + ONE launch for everything else of the solve
                want_l = {0: 6 + 5 * 12 + 1, 1: 6 + 5 * 12 + 1, 2: 6 + 5 * 12 + 2, 3: 8, 4: 2}[mode]
                assert n_l == want_l, (mode, n_l)
                if ref is None:
                    ref = got
                assert got[0] == 12 and np.array_equal(got[2], ref[2]) and np.array_equal(got[3], ref[3]), mode
            else:
                if mode == 0:
                    ref_t = got
                assert got[:2] == ref_t[:2] and np.array_equal(got[2], ref_t[2]) and np.array_equal(got[3], ref_t[3]), mode
    c.t.set_graphs(4)


# ---------------------------------------------------------------- N1: one-end trick loops (Eq. 2.5)
@pytest.mark.parametrize("deriv", [False, True])
def test_one_end_loops_parity_on_the_oracle_solution(small, ragged, deriv):
    """The 16 one-end loops -2ia sum_x s^dag gamma5 Gamma s (appended after the other ops), on the oracle's own
    s: 1e-12 relative to the largest loop; the other ops are unchanged by asking for them."""
    for c in (small, ragged):
        seed = 123
        c.t.loops_reset(deriv, one_end=True)
        rc, _ = c.t.solve(seed, [1, 4], F64, 0.0, 1, slot=0)
        for j, sid in enumerate((1, 4)):
            eta = oracle.noise(c.dims, seed, sid)
            s, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 1e-10, 2000)
            c.t.set_solution(0, j, s)
            want = oracle.all_loops(c.dims, c.theta, c.U, eta, s, deriv, one_end=(c.kappa, c.mu))
            got = c.t.loops_source(0, j)
            assert got.shape == want.shape == (16 + (64 if deriv else 0) + 16, c.dims[3])
            assert rel(got[-16:], want[-16:]) < 1e-12
            assert rel(got[:-16], want[:-16]) < 1e-12
        c.t.loops_reset(False)


def test_one_end_loops_through_eq_2_4(small):
    """Eq. 2.4 on the one-end loops: correction L1(s_HP) - L1(s_LP) plus the LP average, against the oracle's pieces."""
    c = small
    wl = W.WORKLOADS[1]
    got, secs, rc = c.t.run_loop_set(wl.noise_seed, 2, 3, F64, 0.0, 4, hp_tol=1e-10, hp_max_iter=2000, nrhs=2, one_end=True)
    assert rc == 0 and got.shape == (32, c.dims[3])
    corr = np.zeros((32, c.dims[3]), dtype=np.complex128)
    lp = np.zeros_like(corr)
    for j in range(5):
        eta = oracle.noise(c.dims, wl.noise_seed, j)
        s_lp, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 0.0, 4)
        l_lp = oracle.all_loops(c.dims, c.theta, c.U, eta, s_lp, False, one_end=(c.kappa, c.mu))
        if j < 2:
            s_hp, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 1e-10, 2000)
            corr += oracle.all_loops(c.dims, c.theta, c.U, eta, s_hp, False, one_end=(c.kappa, c.mu)) - l_lp
        else:
            lp += l_lp
    want = corr / 2 + lp / 3
    assert rel(got[16:], want[16:]) < 1e-8 and rel(got[:16], want[:16]) < 1e-8
    c.t.loops_reset(False)


def test_one_end_fp32_slot(ragged):
    c = ragged
    c.t.loops_reset(False, one_end=True)
    sols = _oracle_solution_in_fp32_slot(c, 6, [2, 3], 25)
    want = oracle.loops_one_end(c.dims, c.kappa, c.mu, sols[1][1])
    assert rel(c.t.loops_source(1, 1)[16:], want) < 1e-6     # fp32 slot: per-warp sums in fp32, then fp64
    c.t.loops_reset(False)


# ---------------------------------------------------------------- N2: generalised one-end trick loops (Eq. 2.6)
def test_gen_one_end_loops_parity_on_the_oracle_solution(small, ragged):
    """All four operator groups at once (16 local + 64 derivative + 16 one-end + 16 generalised one-end), on the
    oracle's own s: 1e-12 relative to the largest loop of each group."""
    for c in (small, ragged):
        seed = 321
        c.t.loops_reset(True, one_end=True, gen_one_end=True)
        rc, _ = c.t.solve(seed, [0, 5, 9], F64, 0.0, 1, slot=0)
        sols = []
        for j, sid in enumerate((0, 5, 9)):
            eta = oracle.noise(c.dims, seed, sid)
            s, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 1e-10, 2000)
            c.t.set_solution(0, j, s)
            sols.append((eta, s))
        for j, (eta, s) in enumerate(sols):
            want = oracle.all_loops(c.dims, c.theta, c.U, eta, s, True, one_end=(c.kappa, c.mu), gen_one_end=c.kappa)
            got = c.t.loops_source(0, j)
            assert got.shape == want.shape == (112, c.dims[3])
            for lo, hi in ((0, 16), (16, 80), (80, 96), (96, 112)):
                assert rel(got[lo:hi], want[lo:hi]) < 1e-12, (c.dims, j, lo)
        c.t.loops_reset(False)


def test_gen_one_end_alone_and_fp32(ragged):
    c = ragged
    c.t.loops_reset(False, gen_one_end=True)
    sols = _oracle_solution_in_fp32_slot(c, 7, [2, 3], 25)
    want = oracle.loops_gen_one_end(c.dims, c.theta, c.kappa, c.U, sols[0][1])
    got = c.t.loops_source(1, 0)
    assert got.shape == (32, c.dims[3])
    assert rel(got[16:], want) < 1e-5
    c.t.loops_reset(False)


# ---------------------------------------------------------------- N3: momentum-projected loops (reading A25)
MOMENTA = [(0, 0, 0), (1, 0, 0), (0, -1, 0), (0, 0, 1), (1, 1, -1), (-2, 3, 1)]


def test_momentum_loops_parity_on_the_oracle_solution(small, ragged):
    for c in (small, ragged):
        seed = 55
        c.t.loops_reset(True, one_end=True, gen_one_end=True, momenta=MOMENTA)
        rc, _ = c.t.solve(seed, [3, 4], F64, 0.0, 1, slot=0)
        for j, sid in enumerate((3, 4)):
            eta = oracle.noise(c.dims, seed, sid)
            s, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 1e-10, 2000)
            c.t.set_solution(0, j, s)
            want = oracle.all_loops(c.dims, c.theta, c.U, eta, s, True, one_end=(c.kappa, c.mu), gen_one_end=c.kappa,
                                    momenta=MOMENTA)
            got = c.t.loops_source(0, j)
            assert got.shape == want.shape == (112 + 16 * len(MOMENTA), c.dims[3])
            assert rel(got[112:], want[112:]) < 1e-12
            assert rel(got[112:128], got[:16]) < 1e-13             # n = 0 is the local loop (other summation order)
            assert rel(got[:112], want[:112]) < 1e-12
        c.t.loops_reset(False)


def test_momentum_loops_through_eq_2_4_and_fp32(ragged):
    c = ragged
    moms = MOMENTA[1:4]
    got, secs, rc = c.t.run_loop_set(99, 1, 2, F32, 0.0, 6, hp_tol=1e-10, hp_max_iter=2000, nrhs=2, momenta=moms)
    assert rc == 0 and got.shape == (16 + 48, c.dims[3])
    corr = np.zeros_like(got)
    lp = np.zeros_like(got)
    for j in range(3):   # the oracle's own solves: fp64 arithmetic, same iteration counts
        eta = oracle.noise(c.dims, 99, j)
        s_lp, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 0.0, 6)
        l_lp = oracle.all_loops(c.dims, c.theta, c.U, eta, s_lp, False, momenta=moms)
        if j < 1:
            s_hp, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 1e-10, 2000)
            corr += oracle.all_loops(c.dims, c.theta, c.U, eta, s_hp, False, momenta=moms) - l_lp
        else:
            lp += l_lp
    assert rel(got, corr / 1 + lp / 2) < 1e-4          # fp32 LP iterates agree with the fp64 ones to ~2e-5 (A17)
    c.t.loops_reset(False)


# ---------------------------------------------------------------- N4: mixed-precision HP solver
def test_mixed_precision_hp_solve(small, medium, ragged, tsm_mod):
    """fp64 defect correction around the fp32 CG: same solution as the fp64 solve to the accuracy two converged
    solves can agree (A16(iii)): fp64 true residual of the full system <= 1.5e-10, s within 1e-8, loops within
    1e-8; batch independent (A14); tolerance not reached is flagged with the iterate kept."""
    MIXED = tsm_mod.MIXED
    for c, seed in ((small, W.WORKLOADS[1].noise_seed), (medium, W.WORKLOADS[2].noise_seed), (ragged, 17)):
        ids = [1, 6, 2]
        rc, info = c.t.solve(seed, ids, MIXED, 1e-10, 2000, slot=0, want_true_resid=True)
        assert rc == 0, info
        c.t.loops_reset(True)
        for j, sid in enumerate(ids):
            eta = oracle.noise(c.dims, seed, sid)
            s_ref, info_ref = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 1e-10, 2000)
            s = c.t.get_solution(0, j)
            rho = oracle.true_residual(c.dims, c.theta, c.kappa, c.mu, c.U, eta, s)
            assert rho <= 1.5e-10, (c.dims, j, rho)
            assert np.isclose(info[j]["rel_resid_true"], rho, rtol=1e-3)
            assert info[j]["status"] == 0 and info[j]["rel_resid_rec"] <= 1e-10
            assert info_ref["iters"] <= info[j]["iters"] <= 3 * info_ref["iters"]
            assert rel(s, s_ref) < 1e-8
            want = oracle.all_loops(c.dims, c.theta, c.U, eta, s_ref, True)
            assert rel(c.t.loops_source(0, j), want) < 1e-8
        batch = [c.t.get_solution(0, j) for j in range(3)]
        rc, _ = c.t.solve(seed, [ids[1]], MIXED, 1e-10, 2000, slot=1)
        assert np.array_equal(c.t.get_solution(1, 0), batch[1])
        c.t.loops_reset(False)
    c = small
    rc, info = c.t.solve(5, [0], MIXED, 1e-10, 6, slot=0)
    assert rc == tsm_mod.ENOCONV and info[0]["status"] == tsm_mod.ENOCONV and info[0]["rel_resid_rec"] > 1e-10
    with pytest.raises(tsm_mod.TsmError):
        c.t.solve(5, [0], MIXED, 0.0, 10, slot=0)            # needs a tolerance


# ---------------------------------------------------------------- edge cases
@pytest.mark.parametrize("nrhs", [5, 7, 16])
def test_dslash_odd_and_maximum_batch_sizes(tsm_mod, nrhs):
    """Batch sizes that leave source rows of the CTA idle (5, 7) and the maximum (TSM_MAX_NRHS = 16)."""
    c = Case(tsm_mod, (8, 4, 6, 4), 0.6, 91, 0.157, 0.02, -1, max_nrhs=16)
    psi = W.random_spinor(c.dims, 900 + nrhs, nrhs=nrhs)
    for prec, tol in ((F64, 1e-12), (F32, 1e-5)):
        got = _gpu_op(c, 2, prec, psi)
        for j in (0, nrhs // 2, nrhs - 1):
            src = psi[j] if prec == F64 else psi[j].astype(np.complex64).astype(np.complex128)
            assert rel(got[j], _oracle_op(c, 2, src)) < tol, (prec, j)
    rc, info = c.t.solve(3, list(range(nrhs)), F32, 1e-4, 500, slot=1, want_true_resid=True)
    assert rc == 0 and all(i["rel_resid_true"] < 2e-4 for i in info)
    with pytest.raises(tsm_mod.TsmError):
        tsm_mod.Tsm(c.dims, max_nrhs=17)
    c.t.close()


def test_empty_source_sets_and_z2_noise(small):
    """Eq. 2.4 with an empty HP set is Eq. 2.2; with an empty LP set only the correction remains; no sources: zeros."""
    c = small
    seed = 71
    got, _, rc = c.t.run_loop_set(seed, 0, 3, F64, 0.0, 5, nrhs=2)
    assert rc == 0
    want = np.zeros_like(got)
    for j in range(3):
        eta = oracle.noise(c.dims, seed, j)
        s, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 0.0, 5)
        want += oracle.loops(c.dims, eta, s) / 3
    assert rel(got, want) < 1e-12
    got, _, rc = c.t.run_loop_set(seed, 2, 0, F64, 0.0, 5, hp_tol=1e-10, hp_max_iter=2000, nrhs=2)
    corr, lp, n_hp, n_lp = c.t.loops_get_state()
    assert rc == 0 and (n_hp, n_lp) == (2, 0) and not lp.any() and np.array_equal(got, corr / 2)
    got, _, rc = c.t.run_loop_set(seed, 0, 0, F64, 0.0, 5, nrhs=2)
    assert rc == 0 and not got.any()
    # Z2 sources through the solver and the contraction
    rc, info = c.t.solve(seed, [4], F64, 1e-10, 2000, slot=0, kind=1)
    eta = oracle.noise(c.dims, seed, 4, 1)
    assert set(np.unique(eta.real)) == {-1.0, 1.0} and not eta.imag.any()
    s_ref, _ = oracle.solve(c.dims, c.theta, c.kappa, c.mu, c.U, eta, 1e-10, 2000)
    assert rel(c.t.get_solution(0, 0), s_ref) < 1e-11
    c.t.loops_reset(False)
    assert rel(c.t.loops_source(0, 0), oracle.loops(c.dims, eta, s_ref)) < 1e-8


def test_fixed_iterations_far_past_convergence_stay_finite(small):
    """A13: 400 fp64 iterations on a system that converges in ~32: the residual reaches zero / rounding level;
    a source whose <p,Ap> or |r|^2 vanishes is frozen and flagged, never NaN; the solution stays converged."""
    c = small
    rc, info = c.t.solve(8, [0, 1], F64, 0.0, 400, slot=0, want_true_resid=True)
    assert rc in (0, -5)
    for j, i in enumerate(info):
        assert i["status"] in (0, -5) and i["iters"] <= 400
        s = c.t.get_solution(0, j)
        assert np.isfinite(s.view(np.float64)).all()
        assert i["rel_resid_true"] < 1e-12
    rc, info = c.t.solve(8, [0, 1], F32, 0.0, 400, slot=1, want_true_resid=True)
    assert all(np.isfinite(i["rel_resid_true"]) and i["rel_resid_true"] < 1e-5 for i in info)


def test_stencils_write_nothing_outside_their_output(ragged, tsm_mod):
    """compute-sanitizer is closed on this pool: canaries instead.  Output fields sit between guard bands; the
    bands, and the layout padding inside the field (V_h = 720 is padded to 736 sites per source), must be
    untouched by the single-source and the tile kernels (fp64, fp32, bf16; 1, 3 and 12 sources)."""
    import torch
    c = ragged
    Vh = c.t.V // 2
    guard = 4096
    for prec, width in ((F64, 192), (F32, 96), (BF16, 48)):
        for nrhs in (1, 3, 12):
            fb = c.t.field_bytes(prec, nrhs)
            assert fb == width * 736 * nrhs
            src = c.t.pack(prec, W.random_spinor(c.dims, 31, nrhs=nrhs))
            buf = torch.full((guard + 2 * fb + guard,), 0xA5, dtype=torch.uint8, device="cuda")
            out = buf[guard:guard + 2 * fb]
            c.t.dslash(tsm_mod.OP_M_FULL, prec, nrhs, src, out)
            c.t.dslash(tsm_mod.OP_MHAT, prec, nrhs, src[:fb], out[:fb])
            torch.cuda.synchronize()
            assert bool((buf[:guard] == 0xA5).all()) and bool((buf[guard + 2 * fb:] == 0xA5).all()), (prec, nrhs)
            # padding: the last layout block of every source holds 16 live and 16 padding sites
            blk = out[fb:].view(nrhs, 736 // 32, width // 16, 32, 16)
            assert bool((blk[:, -1, :, 16:, :] == 0xA5).all()), (prec, nrhs)
            assert not bool((blk[:, -1, :, :16, :] == 0xA5).all())


@pytest.mark.parametrize("dims", [(16, 16, 4, 4), (8, 32, 4, 4), (32, 8, 4, 6), (64, 4, 4, 4)])
def test_tile_kernel_in_slab_order_on_small_lattices(tsm_mod, dims):
    """Lattices with Lxh * Ly a multiple of 128 take the z-slab tile order (like 32^3 x 64) in k_dslash and
    k_dslash_tile: parity with the oracle and bit-identity of batches with the single-source kernel, fp32 and bf16,
    theta = -1 (the kernels are named explicitly; they are also what the automatic choice picks)."""
    c = Case(tsm_mod, dims, 0.6, 33, 0.157, 0.02, -1, max_nrhs=12)
    psi = W.random_spinor(dims, 77, nrhs=12)
    for nrhs in (3, 5, 12):
        for op in (0, 1, 3):
            c.t.set_stencil_kernel(2)
            got = _gpu_op(c, op, F32, psi[:nrhs])
            for j in (0, nrhs - 1):
                src = psi[j].astype(np.complex64).astype(np.complex128)
                assert rel(got[j], _oracle_op(c, op, src)) < 1e-5, (dims, nrhs, op, j)
                c.t.set_stencil_kernel(1)
                single = _gpu_op(c, op, F32, psi[j:j + 1])[0]
                c.t.set_stencil_kernel(2)
                assert np.array_equal(single, got[j]), (dims, nrhs, op, j)
    for prec in (F32, BF16):
        c.t.set_stencil_kernel(2)
        rc, info = c.t.solve(9, [0, 1, 2, 3, 4], prec, 0.0, 7, slot=0)
        batch = c.t.get_solution(0, 3)
        c.t.set_stencil_kernel(1)
        rc, _ = c.t.solve(9, [3], prec, 0.0, 7, slot=1)
        assert np.array_equal(c.t.get_solution(1, 0), batch), (dims, prec)
    c.t.close()


BOX_LATTICES = [(16, 4, 4, 4),    # Lxh = 8: 4 rows per layout block, one y block (the y halo wraps onto the tile itself)
                (32, 4, 4, 6),    # Lxh = 16 as at 32^3 x 64: 2 rows per block, 2 y blocks, 3 tiles in t
                (64, 4, 6, 4),    # Lxh = 32: one row per block, halo rows are whole blocks
                (8, 8, 4, 4),     # Lxh = 4: 8 rows per block (the shape of config 2)
                (16, 8, 6, 8)]    # 2 y blocks, 3 tiles in z, 4 in t


@pytest.mark.parametrize("theta", [-1, 1])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("dims", BOX_LATTICES)
def test_box_stencil_parity(tsm_mod, dims, recon, theta):
    """k_dslash_box (4-D tiles staged by tensor-map TMA, links in registers; not the automatic choice, see DESIGN.md
    section 6, selected with tsm_set_stencil_kernel): every operator and epilogue form against
    the oracle (1e-5, north_star) on lattices that exercise every halo wrap, for 1, 3 and 12 sources; agreement
    with k_dslash to fp32 rounding; a source's result bit-identical in any batch (A14)."""
    c = Case(tsm_mod, dims, 0.6, 91, 0.157, 0.02, theta, max_nrhs=12, recon=recon)
    assert c.t.stencil_kernel_name(F32, 12) == "k_dslash_small" and c.t.stencil_kernel_name(F32, 1) == "k_dslash_small"   # automatic choice on an L2-resident lattice
    c.t.set_stencil_kernel(3)
    assert c.t.stencil_kernel_name(F32, 12) == "k_dslash_box" and c.t.stencil_kernel_name(F32, 1) == "k_dslash_box"
    assert c.t.stencil_kernel_name(F64, 12) == "k_dslash" and c.t.stencil_kernel_name(BF16, 12) == "k_dslash_tile"
    psi = W.random_spinor(dims, 78, nrhs=12)
    for nrhs in (1, 3, 12):
        for op in (0, 1, 2, 3, 4):
            got = _gpu_op(c, op, F32, psi[:nrhs])
            for j in sorted({0, nrhs - 1}):
                src = psi[j].astype(np.complex64).astype(np.complex128)
                assert rel(got[j], _oracle_op(c, op, src)) < 1e-5, (dims, nrhs, op, j)
            if nrhs > 1:
                single = _gpu_op(c, op, F32, psi[nrhs - 1:nrhs])[0]
                assert np.array_equal(single, got[nrhs - 1]), (dims, nrhs, op)
            if nrhs == 3:
                c.t.set_stencil_kernel(1)
                other = _gpu_op(c, op, F32, psi[:nrhs])
                c.t.set_stencil_kernel(3)
                assert rel(got, other) < 2e-6, (dims, op)
    # through the solver: norm and residual epilogues, CUDA graphs, early exit
    rc, info = c.t.solve(9, [0, 1, 2, 3, 4], F32, 0.0, 7, slot=0, want_true_resid=True)
    batch = c.t.get_solution(0, 3)
    rc, _ = c.t.solve(9, [3], F32, 0.0, 7, slot=1)
    assert np.array_equal(c.t.get_solution(1, 0), batch)
    eta = oracle.noise(dims, 9, 3)
    s_ref, _ = oracle.solve(dims, theta, c.kappa, c.mu, c.U, eta, 0.0, 7)
    assert rel(batch, s_ref) < 2e-5
    rc, info = c.t.solve(9, [5, 6, 7], F32, 1e-4, 500, slot=0, want_true_resid=True)
    assert rc == 0 and all(i["rel_resid_true"] < 2e-4 for i in info)
    c.t.close()


def test_box_stencil_writes_nothing_outside_its_output(tsm_mod):
    import torch
    dims = (32, 4, 4, 6)
    c = Case(tsm_mod, dims, 0.6, 92, 0.157, 0.02, -1, max_nrhs=12)
    c.t.set_stencil_kernel(3)
    guard = 8192
    for nrhs in (1, 5, 12):
        fb = c.t.field_bytes(F32, nrhs)
        src = c.t.pack(F32, W.random_spinor(dims, 31, nrhs=nrhs))
        buf = torch.full((guard + 2 * fb + guard,), 0xA5, dtype=torch.uint8, device="cuda")
        out = buf[guard:guard + 2 * fb]
        c.t.dslash(tsm_mod.OP_M_FULL, F32, nrhs, src, out)
        c.t.dslash(tsm_mod.OP_MHAT_DAG, F32, nrhs, src[:fb], out[:fb])
        torch.cuda.synchronize()
        assert bool((buf[:guard] == 0xA5).all()) and bool((buf[guard + 2 * fb:] == 0xA5).all()), nrhs
        assert np.isfinite(c.t.unpack(F32, nrhs, out).view(np.float64)).all()
    c.t.close()


def test_caller_stream(small, tsm_mod):
    """tsm_set_stream with a caller-owned (non-blocking) torch stream: same results as on the library's own stream,
    including the CUDA-graph replay of the CG iterations on that stream."""
    import torch
    c = small
    rc, info = c.t.solve(11, [0, 1], F32, 0.0, 13, slot=0)
    want = [c.t.get_solution(0, j) for j in range(2)]
    stream = torch.cuda.Stream()
    t2 = tsm_mod.Tsm(c.dims, t_boundary=c.theta, max_nrhs=2, stream=stream)
    t2.set_params(c.kappa, c.mu)
    t2.set_gauge(c.U, 18)
    for _ in range(2):   # the second solve replays cached graphs from the first chunk on
        rc, info2 = t2.solve(11, [0, 1], F32, 0.0, 13, slot=0)
        assert rc == 0 and [i["iters"] for i in info2] == [13, 13]
        for j in range(2):
            assert np.array_equal(t2.get_solution(0, j), want[j])
    t2.loops_reset(True)
    c.t.loops_reset(True)
    assert np.array_equal(t2.loops_source(0, 1), c.t.loops_source(0, 1))
    c.t.loops_reset(False)
    t2.close()


def test_loop_set_is_bit_reproducible(medium):
    """A19: no atomics, fixed reduction trees: the same loop set run twice, and run with another batch size, gives
    bit-identical loops (fp32 LP batches through the tile kernel and CUDA graphs, fp64 and mixed-precision HP)."""
    c = medium
    wl = W.WORKLOADS[2]
    kw = dict(hp_tol=1e-10, hp_max_iter=2000, with_derivative=True, one_end=True)
    c.t.set_hp_precision(0)
    a, _, rc = c.t.run_loop_set(wl.noise_seed, 3, 9, F32, wl.lp_tol, 1000, nrhs=4, **kw)
    b, _, _ = c.t.run_loop_set(wl.noise_seed, 3, 9, F32, wl.lp_tol, 1000, nrhs=4, **kw)
    d, _, _ = c.t.run_loop_set(wl.noise_seed, 3, 9, F32, wl.lp_tol, 1000, nrhs=3, **kw)
    assert rc == 0 and np.array_equal(a, b) and np.array_equal(a, d)
    c.t.set_hp_precision(3)
    e, _, _ = c.t.run_loop_set(wl.noise_seed, 3, 9, F32, wl.lp_tol, 1000, nrhs=4, **kw)
    f, _, _ = c.t.run_loop_set(wl.noise_seed, 3, 9, F32, wl.lp_tol, 1000, nrhs=1, **kw)
    assert np.array_equal(e, f) and rel(e, a) < 1e-8
    c.t.loops_reset(False)


def test_tensor_core_probe_is_correct(small):
    """csrc/mma_probe.cu (the measurement behind DESIGN.md section 6's tensor-core paragraph): every formulation of
    the per-site SU(3) x (3 x 24) product agrees with the fp64 reference it carries -- fp32 FMAs and 3xTF32 to fp32
    rounding, plain TF32 only to ~1e-3 (which is why it cannot serve the 1e-5 stencil), both fp64 forms to 1e-14."""
    for variant, lo, hi in ((0, 0.0, 2e-6), (1, 2e-5, 5e-3), (2, 0.0, 2e-6), (3, 0.0, 1e-14), (4, 0.0, 1e-14)):
        us, err = small.t.probe_su3_tensor(variant, 4096, 8, 2)
        assert us > 0 and lo <= err < hi, (variant, err)


def test_low_precision_only_workspace(small, tsm_mod):
    """tsm_workspace_bytes / tsm_set_workspace with prec = TSM_F32: no fp64 link copy, fp32-sized
    vectors -- fp32 and bf16 solves and their loops are bit-identical to those on the full workspace, noise is still
    bit-exact, fp64 / mixed solves and the fp64 true residual are refused with TSM_ESTATE."""
    c = small
    t2 = tsm_mod.Tsm(c.dims, t_boundary=c.theta, max_nrhs=4, workspace_prec=F32)
    assert t2.workspace.numel() < 0.8 * c.t.workspace.numel()   # 0.59 at 32^3 x 64 with 12 sources; staging weighs more on 4^3 x 8
    t2.set_params(c.kappa, c.mu)
    assert t2.set_gauge(c.U, 18) < 1e-13
    assert np.array_equal(t2.noise(77, 3), oracle.noise(c.dims, 77, 3))
    for prec in (F32, BF16):
        rc, _ = c.t.solve(5, [0, 1, 2], prec, 0.0, 9, slot=1)
        rc2, _ = t2.solve(5, [0, 1, 2], prec, 0.0, 9, slot=1)
        assert rc == 0 and rc2 == 0
        for j in range(3):
            assert np.array_equal(t2.get_solution(1, j), c.t.get_solution(1, j)), (prec, j)
    c.t.loops_reset(True)
    t2.loops_reset(True)
    assert np.array_equal(t2.loops_source(1, 2), c.t.loops_source(1, 2))
    c.t.loops_reset(False)
    for bad in (dict(prec=F64, tol=1e-8), dict(prec=3, tol=1e-8), dict(prec=F32, tol=1e-3, want_true_resid=True)):
        with pytest.raises(tsm_mod.TsmError) as e:
            t2.solve(5, [0], bad["prec"], bad["tol"], 50, slot=0, want_true_resid=bad.get("want_true_resid", False))
        assert e.value.code == tsm_mod.ESTATE, bad
    t2.close()


@pytest.mark.parametrize("recon", [18, 12])
def test_small_lattice_stencil(tsm_mod, recon):
    """k_dslash_small (the automatic choice on lattices of at most 16 384 sites per parity: four warps = four
    directions per 32 sites): every operator and epilogue form against the oracle, fp64 1e-12 and fp32 1e-5, on the
    ragged lattice (last 32-site block half empty) for 1, 3 and 12 sources; agreement with k_dslash to rounding
    (the sum over directions is associated differently); a source's result bit-identical in any batch (A14); and
    through the solver (norm and residual epilogues, graphs), fp64 iterates at equal iteration count to 1e-12."""
    dims, theta = (6, 10, 4, 6), +1
    c = Case(tsm_mod, dims, 0.6, 77, 0.157, 0.02, theta, max_nrhs=12, recon=recon)
    assert c.t.stencil_kernel_name(F64, 1) == "k_dslash_small" and c.t.stencil_kernel_name(BF16, 4) == "k_dslash_tile"
    psi = W.random_spinor(dims, 80, nrhs=12)
    for prec, tol, close in ((F64, 1e-12, 1e-14), (F32, 1e-5, 2e-6)):
        for nrhs in (1, 3, 12):
            for op in (0, 1, 2, 3, 4):
                got = _gpu_op(c, op, prec, psi[:nrhs])
                for j in sorted({0, nrhs - 1}):
                    src = psi[j] if prec == F64 else psi[j].astype(np.complex64).astype(np.complex128)
                    assert rel(got[j], _oracle_op(c, op, src)) < tol, (prec, nrhs, op, j)
                if nrhs == 12:
                    single = _gpu_op(c, op, prec, psi[5:6])[0]
                    assert np.array_equal(single, got[5]), (prec, op)
                if nrhs == 3:
                    c.t.set_stencil_kernel(1)
                    other = _gpu_op(c, op, prec, psi[:nrhs])
                    c.t.set_stencil_kernel(0)
                    assert rel(got, other) < close, (prec, op)
    eta = oracle.noise(dims, 9, 3)
    for k in (1, 4, 9):
        s_ref, _ = oracle.solve(dims, theta, c.kappa, c.mu, c.U, eta, 0.0, k)
        rc, info = c.t.solve(9, [1, 2, 3, 4], F64, 0.0, k, slot=0)
        assert rc == 0 and rel(c.t.get_solution(0, 2), s_ref) < 1e-12, k
    rc, info = c.t.solve(9, [0, 1, 2, 3, 4], F32, 0.0, 7, slot=0)
    batch = c.t.get_solution(0, 3)
    rc, _ = c.t.solve(9, [3], F32, 0.0, 7, slot=1)
    assert np.array_equal(c.t.get_solution(1, 0), batch)
    rc, info = c.t.solve(9, [5, 6, 7], F32, 1e-4, 500, slot=0, want_true_resid=True)
    assert rc == 0 and all(i["rel_resid_true"] < 2e-4 for i in info)
    c.t.close()


def test_async_solves_match_synchronous_ones(medium, tsm_mod):
    """tsm_solve_async + tsm_solve_wait: the same iterates, iteration counts and statuses as tsm_solve, bit for bit, in
    fixed-iteration and residual mode (there the stopping test runs on the device), with the next solve enqueued
    before the first is waited for; the Eq. 2.4 set (whose LP-only batches are enqueued the same way) is unchanged;
    waiting on a slot with nothing pending is an error."""
    c = medium
    for prec, tol, k in ((F32, 0.0, 11), (F32, 1e-4, 500), (F64, 1e-9, 2000), (BF16, 5e-3, 200)):
        rc, info = c.t.solve(21, [0, 1, 2], prec, tol, k, slot=0)
        want = [c.t.get_solution(0, j) for j in range(3)]
        c.t.solve_async(21, [0, 1, 2], prec, tol, k, slot=1)
        c.t.loops_reset(False)
        c.t.loops_add_lp(1)                                  # uses the slot on the stream, no wait in between
        c.t.solve_async(21, [7, 8, 9], prec, tol, k, slot=0)   # and the next solve is already enqueued
        rc2, info2 = c.t.solve_wait(1)
        assert rc2 == rc and [i["iters"] for i in info2] == [i["iters"] for i in info], (prec, tol)
        assert [i["status"] for i in info2] == [i["status"] for i in info]
        for j in range(3):
            assert np.array_equal(c.t.get_solution(1, j), want[j]), (prec, tol, j)
        rc3, info3 = c.t.solve_wait(0)
        assert rc3 == 0 and len(info3) == 3
    with pytest.raises(tsm_mod.TsmError) as e:
        c.t.solve_wait(0)
    assert e.value.code == tsm_mod.ESTATE
    c.t.loops_reset(False)


@pytest.mark.parametrize("stencil", [1, 0])
@pytest.mark.parametrize("dims,recon", [((8, 8, 8, 16), 18), ((6, 10, 4, 6), 18), ((16, 16, 16, 32), 12), ((4, 4, 4, 8), 18)])
def test_persistent_cg_kernel(tsm_mod, dims, recon, stencil):
    """tsm_set_graphs(3): the whole CG loop in one cooperative launch of k_cg_persistent (grid barriers between the
    phases, dot products summed from per-tile partials by every CTA, stopping test on the device).  Its phases are the
    code of the kernel-by-kernel path, so with k_dslash as the stencil of that path (forced where k_dslash_small would
    be chosen) the iterates are BIT-identical: fixed-iteration and residual mode, fp64 and fp32, 1, 3 and 4 sources,
    a batch whose sources stop at different iterations, and the mixed-precision HP solver on top of it; fp64 also
    against the oracle at 1e-12 and by true residual.  stencil = 0: the automatic choice -- on lattices of at most
    16 384 sites per parity that is k_dslash_small, and the persistent kernel is then k_cg_persistent_small (the same
    loop with small_block() as the stencil), again bit-identical to its kernel-by-kernel path."""
    c = Case(tsm_mod, dims, 0.5, 57, 0.157, 0.01, -1, max_nrhs=4, recon=recon)
    c.t.set_stencil_kernel(stencil)
    seed = 99
    cases = [(F64, 0.0, 9, [1, 2, 3]), (F32, 0.0, 13, [4]), (F32, 1e-4, 500, [5, 6, 7, 8]), (F64, 1e-9, 2000, [2, 9]), (3, 1e-10, 2000, [1, 2, 3])]
    ref = {}
    for mode in (0, 3, 4):   # 4: automatic -- where k_dslash_small is the stencil, the whole solve after the noise is one launch
        c.t.set_graphs(mode)
        for k, (prec, tol, it, ids) in enumerate(cases):
            n0 = c.t.launch_count()
            rc, info = c.t.solve(seed, ids, prec, tol, it, slot=0, want_true_resid=(prec != F32))
            got = ([i["iters"] for i in info], [i["status"] for i in info], [c.t.get_solution(0, j) for j in range(len(ids))])
            if mode == 0:
                ref[k] = got
            else:
                assert rc == 0 and got[0] == ref[k][0] and got[1] == ref[k][1], (dims, k, got[0], ref[k][0])
                for j in range(len(ids)):
                    assert np.array_equal(got[2][j], ref[k][2][j]), (dims, k, j)
            if prec != F32 and tol > 0:
                assert all(i["rel_resid_true"] < 20 * tol for i in info), (dims, k)
    eta = oracle.noise(dims, seed, 2)
    s_ref, _ = oracle.solve(dims, -1, c.kappa, c.mu, c.U, eta, 0.0, 9)
    c.t.set_graphs(3)
    rc, info = c.t.solve(seed, [1, 2, 3], F64, 0.0, 9, slot=0)
    assert rel(c.t.get_solution(0, 1), s_ref) < 1e-12
    # a single launch for the loop: noise, twist, 3 stencils, init, ONE persistent launch, reconstruction
    n0 = c.t.launch_count()
    c.t.solve(seed, [4], F32, 0.0, 13, slot=0)
    assert c.t.launch_count() - n0 == 6 + 1 + 1
    # automatic mode, solves only enqueued (tsm_solve_async): the same iterates as the kernel-by-kernel path, against
    # the oracle too; where the one-launch solve applies a batch is the noise kernel plus ONE launch
    c.t.set_graphs(4)
    for k in (0, 2, 3):
        prec, tol, it, ids = cases[k]
        n0 = c.t.launch_count()
        c.t.solve_async(seed, ids, prec, tol, it, slot=1)
        n_l = c.t.launch_count() - n0
        rc, info = c.t.solve_wait(1)
        assert rc == 0 and [i["iters"] for i in info] == ref[k][0], (dims, k)
        for j in range(len(ids)):
            assert np.array_equal(c.t.get_solution(1, j), ref[k][2][j]), (dims, k, j)
        if stencil == 0 and dims[0] * dims[1] * dims[2] * dims[3] // 2 <= 16384:
            assert n_l == 2, (dims, k, n_l)
    if dims[3] <= 16:   # (the oracle's converged solve of the largest lattice here would take a minute)
        s_conv, _ = oracle.solve(dims, -1, c.kappa, c.mu, c.U, oracle.noise(dims, seed, 2), 1e-9, 2000)
        assert rel(c.t.get_solution(1, 0), s_conv) < 1e-6
    c.t.close()
