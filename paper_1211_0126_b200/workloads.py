"""Seeded synthetic inputs and the five BASELINE.json workloads.

This module holds NO arithmetic of the method (no Dirac operator, no gamma
matrices, no noise generator, no solver).  It only produces the *inputs* that
both the CPU oracle (oracle/) and the CUDA path consume: SU(3) gauge links and
the table of workload parameters.  It imports neither of them.

The paper measured on the ETMC B55 ensemble (32^3 x 64, section 3);
those gauge configurations are not available, so seeded random SU(3) links of
the same shape stand in (reading A21; recipe restated in
DESIGN.md "Input recipe").
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field

import numpy as np

# Gell-Mann matrices lambda_1..lambda_8 (standard normalisation tr(l_a l_b) = 2 delta_ab).
_GELL_MANN = np.zeros((8, 3, 3), dtype=np.complex128)
_GELL_MANN[0][0, 1] = _GELL_MANN[0][1, 0] = 1
_GELL_MANN[1][0, 1] = -1j
_GELL_MANN[1][1, 0] = 1j
_GELL_MANN[2][0, 0] = 1
_GELL_MANN[2][1, 1] = -1
_GELL_MANN[3][0, 2] = _GELL_MANN[3][2, 0] = 1
_GELL_MANN[4][0, 2] = -1j
_GELL_MANN[4][2, 0] = 1j
_GELL_MANN[5][1, 2] = _GELL_MANN[5][2, 1] = 1
_GELL_MANN[6][1, 2] = -1j
_GELL_MANN[6][2, 1] = 1j
_GELL_MANN[7][0, 0] = _GELL_MANN[7][1, 1] = 1 / np.sqrt(3.0)
_GELL_MANN[7][2, 2] = -2 / np.sqrt(3.0)


def volume(dims) -> int:
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def random_su3_links(dims, eps: float, seed: int, chunk: int = 1 << 16) -> np.ndarray:
    """Seeded weak-field SU(3) links U = exp(i*eps*H).

    H = sum_a c_a lambda_a / 2 with c_a uniform in [-1, 1) (reading A21), drawn
    from numpy's PCG64 stream `seed` in the order [mu][lex][a].  exp() is taken
    through the Hermitian eigendecomposition of H.  Returns a complex128 array
    of shape [4][V][3][3] (row-major colour indices, lex = x + Lx*(y + Ly*(z + Lz*t))).
    """
    V = volume(dims)
    rng = np.random.Generator(np.random.PCG64(seed))
    n = 4 * V
    out = np.empty((n, 3, 3), dtype=np.complex128)
    gm = _GELL_MANN.reshape(8, 9)
    # the random stream is drawn serially in [mu][lex][a] order; only the per-matrix
    # eigendecompositions run on a thread pool, so the result does not depend on the pool size
    coef = rng.random((n, 8)) * 2.0 - 1.0

    def work(lo):
        hi = min(n, lo + chunk)
        H = (coef[lo:hi] @ gm).reshape(hi - lo, 3, 3) * 0.5
        w, v = np.linalg.eigh(H)
        out[lo:hi] = (v * np.exp(1j * eps * w)[:, None, :]) @ v.conj().transpose(0, 2, 1)

    starts = range(0, n, chunk)
    nthreads = min(len(os.sched_getaffinity(0)), 16, len(starts))
    if nthreads > 1:
        with ThreadPoolExecutor(nthreads) as ex:
            list(ex.map(work, starts))
    else:
        for lo in starts:
            work(lo)
    return out.reshape(4, V, 3, 3)


def unit_links(dims) -> np.ndarray:
    """Free field U = 1 (for closed-form momentum-space checks)."""
    V = volume(dims)
    out = np.zeros((4, V, 3, 3), dtype=np.complex128)
    out[..., 0, 0] = out[..., 1, 1] = out[..., 2, 2] = 1.0
    return out


def random_su3_sites(dims, seed: int) -> np.ndarray:
    """One Haar-ish random SU(3) matrix per site, [V][3][3] (gauge transforms)."""
    V = volume(dims)
    rng = np.random.Generator(np.random.PCG64(seed))
    z = rng.standard_normal((V, 3, 3)) + 1j * rng.standard_normal((V, 3, 3))
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=1, axis2=2)
    q = q * (d / np.abs(d))[:, None, :]
    det = np.linalg.det(q)
    q[:, :, 2] *= (1.0 / det)[:, None]
    return q


def gauge_transform(dims, U: np.ndarray, Om: np.ndarray) -> np.ndarray:
    """U'_mu(x) = Omega(x) U_mu(x) Omega(x+mu)^dagger (periodic shift of the site index)."""
    Lx, Ly, Lz, Lt = (int(d) for d in dims)
    V = Lx * Ly * Lz * Lt
    idx = np.arange(V).reshape(Lt, Lz, Ly, Lx)
    out = np.empty_like(U)
    for mu, ax in enumerate((3, 2, 1, 0)):
        fwd = np.roll(idx, -1, axis=ax).reshape(-1)
        out[mu] = np.einsum("nij,njk,nlk->nil", Om, U[mu], Om[fwd].conj())
    return out


def average_plaquette(dims, U: np.ndarray) -> float:
    """(1/3) Re tr of the plaquette, averaged over sites and the 6 planes (logged only)."""
    Lx, Ly, Lz, Lt = (int(d) for d in dims)
    V = Lx * Ly * Lz * Lt
    idx = np.arange(V).reshape(Lt, Lz, Ly, Lx)
    axes = (3, 2, 1, 0)
    fwd = [np.roll(idx, -1, axis=ax).reshape(-1) for ax in axes]
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            p = np.einsum("nij,njk,nlk,nml->nim", U[mu], U[nu][fwd[mu]],
                          U[mu][fwd[nu]].conj(), U[nu].conj())
            tot += np.trace(p, axis1=1, axis2=2).real.mean() / 3.0
    return tot / 6.0


def random_spinor(dims, seed: int, nrhs: int | None = None) -> np.ndarray:
    """Seeded Gaussian spinor field [V][4][3] complex128 (operator test vectors)."""
    V = volume(dims)
    rng = np.random.Generator(np.random.PCG64(seed))
    shape = (V, 4, 3) if nrhs is None else (nrhs, V, 4, 3)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


@dataclass(frozen=True)
class Workload:
    """One row of SURVEY.md section 8d (BASELINE.json `configs`, readings A10/A11)."""
    name: str
    dims: tuple
    eps: float
    kappa: float
    mu: float
    lp_prec: str            # "f64" | "f32" | "bf16"
    lp_tol: float           # 0 => fixed-iteration truncation
    lp_iters: int           # iteration cap (fixed count when lp_tol == 0)
    hp_tol: float
    n_hp: int
    n_lp: int
    nrhs: int
    reconstruct: int        # 18 | 12 (low-precision link storage)
    derivative: bool
    t_boundary: int = -1    # reading A3
    gauge_seed: int = 0
    noise_seed: int = 0
    extra: dict = field(default_factory=dict)

    @property
    def V(self) -> int:
        return volume(self.dims)

    def links(self) -> np.ndarray:
        return random_su3_links(self.dims, self.eps, self.gauge_seed)


def _wl(i, **kw):
    return Workload(gauge_seed=12110126 + i, noise_seed=0x1211012600000000 + i, **kw)


WORKLOADS = {
    1: _wl(1, name="cfg1_4x4x4x8", dims=(4, 4, 4, 8), eps=0.2, kappa=0.15, mu=0.01,
           lp_prec="f64", lp_tol=1e-2, lp_iters=1000, hp_tol=1e-10, n_hp=2, n_lp=4,
           nrhs=1, reconstruct=18, derivative=False),
    2: _wl(2, name="cfg2_8x8x8x16", dims=(8, 8, 8, 16), eps=0.2, kappa=0.155, mu=0.005,
           lp_prec="f32", lp_tol=1e-3, lp_iters=1000, hp_tol=1e-10, n_hp=4, n_lp=16,
           nrhs=1, reconstruct=18, derivative=False),
    3: _wl(3, name="cfg3_16x16x16x32", dims=(16, 16, 16, 32), eps=0.5, kappa=0.158, mu=0.004,
           lp_prec="f32", lp_tol=0.0, lp_iters=50, hp_tol=1e-10, n_hp=8, n_lp=64,
           nrhs=1, reconstruct=12, derivative=False),
    4: _wl(4, name="cfg4_24x24x24x48", dims=(24, 24, 24, 48), eps=0.7, kappa=0.1605, mu=0.0035,
           lp_prec="bf16", lp_tol=5e-3, lp_iters=1000, hp_tol=1e-10, n_hp=16, n_lp=200,
           nrhs=4, reconstruct=12, derivative=False),
    5: _wl(5, name="cfg5_32x32x32x64", dims=(32, 32, 32, 64), eps=0.7, kappa=0.161236, mu=0.0055,
           lp_prec="f32", lp_tol=0.0, lp_iters=100, hp_tol=1e-10, n_hp=24, n_lp=500,
           nrhs=12, reconstruct=18, derivative=True),
}
