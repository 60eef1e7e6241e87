"""TEST INFRASTRUCTURE: ctypes front end of the fp64 CPU oracle (oracle/tsm_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_1211_0126_b200 (the CUDA
path), and the CUDA path never imports it.

All arrays are numpy complex128 in the host layouts of SURVEY.md 8(c) C1-C2:
spinor [V][4][3], links [4][V][3][3], loops [n_ops][Lt].

The TSM combination (Eq. 2.4, readings A10/A11, O7) is written
here in plain Python on top of the C pieces so it can be read against the paper.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tsm_oracle.c")
_LIB = os.path.join(_HERE, "libtsm_oracle.so")
_lib = None

_c_int4 = ctypes.c_int * 4
_dp = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 -fopenmp."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=c11", "-shared", "-fPIC",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_true_residual.restype = ctypes.c_double
    return _lib


def _d(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def _c128(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.complex128)


def n_threads() -> int:
    """Threads the OpenMP site loop will use (OMP_NUM_THREADS or the affinity mask)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        return int(env.split(",")[0])
    return len(os.sched_getaffinity(0))


def gamma(idx: int) -> np.ndarray:
    out = np.zeros((4, 4), dtype=np.complex128)
    lib().oracle_gamma(ctypes.c_int(idx), _d(out))
    return out


def philox4x32_10(ctr, key) -> np.ndarray:
    c = (ctypes.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (ctypes.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (ctypes.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return np.array(list(o), dtype=np.uint32)


def noise(dims, seed: int, source_id: int, kind: int = 0) -> np.ndarray:
    V = int(np.prod(dims))
    out = np.empty((V, 4, 3), dtype=np.complex128)
    lib().oracle_noise(_c_int4(*dims), ctypes.c_uint64(seed), ctypes.c_uint32(source_id),
                       ctypes.c_int(kind), _d(out))
    return out


def hop(dims, theta: int, U, psi, parity: int = -1) -> np.ndarray:
    U = _c128(U)
    psi = _c128(psi)
    out = np.empty_like(psi)
    lib().oracle_hop(_c_int4(*dims), ctypes.c_int(theta), _d(U), _d(psi), _d(out), ctypes.c_int(parity))
    return out


def _apply(fn, dims, theta, kappa, mu, U, psi):
    U = _c128(U)
    psi = _c128(psi)
    out = np.empty_like(psi)
    fn(_c_int4(*dims), ctypes.c_int(theta), ctypes.c_double(kappa), ctypes.c_double(mu),
       _d(U), _d(psi), _d(out))
    return out


def apply_M(dims, theta, kappa, mu, U, psi) -> np.ndarray:
    return _apply(lib().oracle_apply_M, dims, theta, kappa, mu, U, psi)


def apply_Mhat(dims, theta, kappa, mu, U, psi_even) -> np.ndarray:
    """psi_even: full-lattice array that is zero on odd sites."""
    return _apply(lib().oracle_apply_Mhat, dims, theta, kappa, mu, U, psi_even)


def apply_Mhat_dag(dims, theta, kappa, mu, U, psi_even) -> np.ndarray:
    return _apply(lib().oracle_apply_Mhat_dag, dims, theta, kappa, mu, U, psi_even)


def solve(dims, theta, kappa, mu, U, eta, tol: float, max_iter: int):
    """Returns (s, info) with info = dict(iters, rel_resid_rec, rel_resid_true, status)."""
    U = _c128(U)
    eta = _c128(eta)
    s = np.empty_like(eta)
    info = np.zeros(4, dtype=np.float64)
    lib().oracle_solve(_c_int4(*dims), ctypes.c_int(theta), ctypes.c_double(kappa),
                       ctypes.c_double(mu), _d(U), _d(eta), ctypes.c_double(tol),
                       ctypes.c_int(max_iter), _d(s), _d(info))
    return s, dict(iters=int(info[0]), rel_resid_rec=float(info[1]),
                   rel_resid_true=float(info[2]), status=int(info[3]))


def true_residual(dims, theta, kappa, mu, U, eta, s) -> float:
    U = _c128(U)
    eta = _c128(eta)
    s = _c128(s)
    return float(lib().oracle_true_residual(_c_int4(*dims), ctypes.c_int(theta),
                                            ctypes.c_double(kappa), ctypes.c_double(mu),
                                            _d(U), _d(eta), _d(s)))


def loops(dims, eta, s) -> np.ndarray:
    eta = _c128(eta)
    s = _c128(s)
    out = np.empty((16, dims[3]), dtype=np.complex128)
    lib().oracle_loops(_c_int4(*dims), _d(eta), _d(s), _d(out))
    return out


def cov_diff(dims, theta, U, mu_dir: int, s) -> np.ndarray:
    U = _c128(U)
    s = _c128(s)
    out = np.empty_like(s)
    lib().oracle_cov_diff(_c_int4(*dims), ctypes.c_int(theta), _d(U), ctypes.c_int(mu_dir), _d(s), _d(out))
    return out


def loops_deriv(dims, theta, U, eta, s) -> np.ndarray:
    U = _c128(U)
    eta = _c128(eta)
    s = _c128(s)
    out = np.empty((4, 16, dims[3]), dtype=np.complex128)
    lib().oracle_loops_deriv(_c_int4(*dims), ctypes.c_int(theta), _d(U), _d(eta), _d(s), _d(out))
    return out


def loops_one_end(dims, kappa, mu, s) -> np.ndarray:
    """Eq. 2.5: per-source one-end loops -2ia sum_x s^dag gamma5 Gamma s, [16][Lt]."""
    s = _c128(s)
    out = np.empty((16, dims[3]), dtype=np.complex128)
    lib().oracle_loops_one_end(_c_int4(*dims), ctypes.c_double(kappa), ctypes.c_double(mu), _d(s), _d(out))
    return out


def loops_gen_one_end(dims, theta, kappa, U, s) -> np.ndarray:
    """Eq. 2.6: per-source generalised one-end loops 2 sum_x s^dag g5 Gamma g5 D_W s, [16][Lt]."""
    U = _c128(U)
    s = _c128(s)
    out = np.empty((16, dims[3]), dtype=np.complex128)
    lib().oracle_loops_gen_one_end(_c_int4(*dims), ctypes.c_int(theta), ctypes.c_double(kappa), _d(U), _d(s), _d(out))
    return out


def loops_momentum(dims, eta, s, momenta) -> np.ndarray:
    """Reading A25: L_Gamma(t, p) = sum_x exp(+i p.x) eta^dag Gamma s, p_i = 2 pi n_i / L_i; [nmom][16][Lt]."""
    eta = _c128(eta)
    s = _c128(s)
    mom = np.ascontiguousarray(momenta, dtype=np.int32).reshape(-1, 3)
    out = np.empty((mom.shape[0], 16, dims[3]), dtype=np.complex128)
    lib().oracle_loops_momentum(_c_int4(*dims), _d(eta), _d(s), ctypes.c_int(mom.shape[0]),
                                mom.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), _d(out))
    return out


def all_loops(dims, theta, U, eta, s, with_derivative: bool, one_end=None, gen_one_end=None, momenta=None) -> np.ndarray:
    """[n_ops][Lt]: the 16 local loops, then (if asked) [mu][Gamma] derivative loops (O6b order), then
    (if one_end=(kappa, mu) is given) the 16 one-end loops of Eq. 2.5, then (if gen_one_end=kappa is given)
    the 16 generalised one-end loops of Eq. 2.6, then (if momenta [nmom][3] are given) 16 momentum-projected
    local loops per momentum (reading A25)."""
    parts = [loops(dims, eta, s)]
    if with_derivative:
        parts.append(loops_deriv(dims, theta, U, eta, s).reshape(64, dims[3]))
    if one_end is not None:
        parts.append(loops_one_end(dims, one_end[0], one_end[1], s))
    if gen_one_end is not None:
        parts.append(loops_gen_one_end(dims, theta, gen_one_end, U, s))
    if momenta is not None:
        parts.append(loops_momentum(dims, eta, s, momenta).reshape(-1, dims[3]))
    return parts[0] if len(parts) == 1 else np.concatenate(parts, axis=0)


def tsm_loops(dims, theta, kappa, mu, U, seed, n_hp, n_lp, hp_tol, hp_max_iter,
              lp_tol, lp_max_iter, with_derivative=False, kind=0, per_source=None):
    """Eq. 2.4 on loops, reading O7 / A10:

    L_TSM = (1/N_HP) sum_{j<N_HP} [L(eta_j, s_j^HP) - L(eta_j, s_j^LP)]
          + (1/N_LP) sum_{N_HP <= j < N_HP+N_LP} L(eta_j, s_j^LP)

    Sources j = 0..N_HP-1 get an HP and an LP solve of the same eta_j; sources
    j = N_HP..N_HP+N_LP-1 get an LP solve only.  `per_source`, if a dict, receives
    the per-source loops and solve infos.
    """
    n_ops = 16 + (64 if with_derivative else 0)
    corr = np.zeros((n_ops, dims[3]), dtype=np.complex128)
    lp_sum = np.zeros((n_ops, dims[3]), dtype=np.complex128)
    for j in range(n_hp):
        eta = noise(dims, seed, j, kind)
        s_hp, info_hp = solve(dims, theta, kappa, mu, U, eta, hp_tol, hp_max_iter)
        s_lp, info_lp = solve(dims, theta, kappa, mu, U, eta, lp_tol, lp_max_iter)
        l_hp = all_loops(dims, theta, U, eta, s_hp, with_derivative)
        l_lp = all_loops(dims, theta, U, eta, s_lp, with_derivative)
        corr += l_hp - l_lp
        if per_source is not None:
            per_source[j] = dict(hp=l_hp, lp=l_lp, info_hp=info_hp, info_lp=info_lp)
    for j in range(n_hp, n_hp + n_lp):
        eta = noise(dims, seed, j, kind)
        s_lp, info_lp = solve(dims, theta, kappa, mu, U, eta, lp_tol, lp_max_iter)
        l_lp = all_loops(dims, theta, U, eta, s_lp, with_derivative)
        lp_sum += l_lp
        if per_source is not None:
            per_source[j] = dict(lp=l_lp, info_lp=info_lp)
    out = np.zeros_like(corr)
    if n_hp > 0:
        out += corr / n_hp
    if n_lp > 0:
        out += lp_sum / n_lp
    return out
