"""FP64 CPU oracle for the real-space AMOEBA polarization hot path.

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package; the CUDA product
(``paper_2011_01207_b200``) never does, and nothing here imports the product.

The pair arithmetic lives in ``tkhp_oracle.c`` (plain C, O(N^2) minimum-image
double loops, see its header for the citations).  This file holds

* the ctypes loader/builder for that C file (``gcc -O2 -fopenmp
  -ffp-contract=off``, no ``-ffast-math``);
* (S) the PCG solve, written step by step in the order of SURVEY.md 8(c) "S"
  (paper: "conjugate gradient solver and a diagonal preconditioner", PAPER.md
  L437; one matrix-vector product per iteration, L160);
* the dense reference solve A mu = E by Cholesky (library primitive) for small N;
* (U) the polarization energy;
* (N) the checks on a neighbour list handed over by the library: permutation
  validity, sort-key order, block boxes and the brute-force block-pair set.

Every function cites the passage it follows.  Pins: tests/test_oracle_*.py.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

__all__ = [
    "build", "lib", "ewald_bn", "thole_lambda", "pair_G", "perm_field",
    "perm_field_rows", "tmatvec", "tmatvec_rows", "dense_T", "dense_A",
    "count_pairs", "count_pairs_rows", "pcg_solve", "dense_solve",
    "polar_energy", "COULOMB", "wrap", "grid_bits", "cell_coords",
    "hilbert_key", "sort_keys", "check_perm", "block_boxes", "block_pairs",
    "atom_pairs_covered", "num_threads", "to_fixed", "from_fixed", "FIX_VEC_BITS", "FIX_ENERGY_BITS",
    "polar_energy_fixed",
    "OPEN_MAX_BITS",
]

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "tkhp_oracle.c"
_SO = _HERE / "libtkhp_oracle.so"

COULOMB = 332.063713  # kcal*A/(mol*e^2), SURVEY 8(c) U / Q12

_lib = None
_f64p = ctypes.POINTER(ctypes.c_double)
_i32p = ctypes.POINTER(ctypes.c_int32)
_i64p = ctypes.POINTER(ctypes.c_int64)


def build(force: bool = False) -> Path:
    """Compile tkhp_oracle.c into oracle/libtkhp_oracle.so (in-tree, git-ignored)."""
    if force or not _SO.exists() or _SO.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _SO.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC",
               "-shared", "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _SO)
    return _SO


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(str(_SO))
        d, i64 = ctypes.c_double, ctypes.c_int64
        L.oracle_ewald_bn.argtypes = [d, d, _f64p]
        L.oracle_ewald_bn.restype = None
        L.oracle_thole_lambda.argtypes = [d, d, d, d, _f64p]
        L.oracle_thole_lambda.restype = None
        L.oracle_pair_G.argtypes = [d, d, d, d, d, d, _f64p]
        L.oracle_pair_G.restype = None
        L.oracle_perm_field.argtypes = [i64, _f64p, _f64p, _f64p, _f64p, _f64p, _i32p,
                                        d, d, d, d, _f64p]
        L.oracle_perm_field_rows.argtypes = [i64, _f64p, _f64p, _f64p, _f64p, _f64p, _i32p,
                                             d, d, d, d, i64, _i64p, _f64p]
        L.oracle_tmatvec.argtypes = [i64, _f64p, _f64p, _f64p, d, d, d, d, _f64p]
        L.oracle_tmatvec_rows.argtypes = [i64, _f64p, _f64p, _f64p, d, d, d, d,
                                          i64, _i64p, _f64p]
        L.oracle_dense_T.argtypes = [i64, _f64p, _f64p, d, d, d, d, _f64p]
        L.oracle_count_pairs.argtypes = [i64, _f64p, d, d]
        L.oracle_count_pairs.restype = i64
        L.oracle_count_pairs_rows.argtypes = [i64, _f64p, d, d, i64, _i64p]
        L.oracle_count_pairs_rows.restype = i64
        L.oracle_wrap.argtypes = [d, d]
        L.oracle_wrap.restype = d
        L.oracle_block_boxes.argtypes = [i64, _i32p, _f64p, d, _f64p, _f64p]
        L.oracle_block_pairs.argtypes = [i64, _f64p, _f64p, d, d, _i32p, i64]
        L.oracle_block_pairs.restype = i64
        _lib = L
    return _lib


def num_threads() -> int:
    """Threads the OpenMP loops use (OMP_NUM_THREADS or all cores)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        return int(env.split(",")[0])
    return len(os.sched_getaffinity(0))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t=_f64p):
    return a.ctypes.data_as(t)


# ------------------------------------------------------------ radial functions
def ewald_bn(beta: float, R: float) -> np.ndarray:
    """bn_0..bn_3 (SURVEY 8(c) "Radial functions", Ewald)."""
    out = np.zeros(4)
    lib().oracle_ewald_bn(beta, R, _p(out))
    return out


def thole_lambda(a: float, alpha_i: float, alpha_j: float, R: float) -> np.ndarray:
    """lambda_3, lambda_5, lambda_7 (SURVEY 8(c) "Radial functions", Thole)."""
    out = np.zeros(3)
    lib().oracle_thole_lambda(a, alpha_i, alpha_j, R, _p(out))
    return out


def pair_G(beta, a, alpha_i, alpha_j, s, R) -> np.ndarray:
    """G_1..G_3 of (F1)."""
    out = np.zeros(3)
    lib().oracle_pair_G(beta, a, alpha_i, alpha_j, float(s), R, _p(out))
    return out


# ------------------------------------------------------------------ F, T
def perm_field(sys_) -> np.ndarray:
    """(F1-F3) permanent-multipole field at every atom, (N,3)."""
    n = sys_.n_atoms
    E = np.zeros((n, 3))
    pos, q, dip, quad, al = map(_f64, (sys_.pos, sys_.charge, sys_.dipole, sys_.quad,
                                       sys_.polarizability))
    g = np.ascontiguousarray(sys_.group_id, dtype=np.int32)
    lib().oracle_perm_field(n, _p(pos), _p(q), _p(dip), _p(quad), _p(al), _p(g, _i32p),
                            sys_.box, sys_.cutoff, sys_.ewald_beta, sys_.thole_a, _p(E))
    return E


def perm_field_rows(sys_, rows) -> np.ndarray:
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    E = np.zeros((rows.size, 3))
    pos, q, dip, quad, al = map(_f64, (sys_.pos, sys_.charge, sys_.dipole, sys_.quad,
                                       sys_.polarizability))
    g = np.ascontiguousarray(sys_.group_id, dtype=np.int32)
    lib().oracle_perm_field_rows(sys_.n_atoms, _p(pos), _p(q), _p(dip), _p(quad), _p(al),
                                 _p(g, _i32p), sys_.box, sys_.cutoff, sys_.ewald_beta,
                                 sys_.thole_a, rows.size, _p(rows, _i64p), _p(E))
    return E


def tmatvec(sys_, mu) -> np.ndarray:
    """(T1,T2) out = T_real mu + self mu, (N,3)."""
    n = sys_.n_atoms
    mu = _f64(mu).reshape(n, 3)
    out = np.zeros((n, 3))
    pos, al = _f64(sys_.pos), _f64(sys_.polarizability)
    lib().oracle_tmatvec(n, _p(pos), _p(al), _p(mu), sys_.box, sys_.cutoff,
                         sys_.ewald_beta, sys_.thole_a, _p(out))
    return out


def tmatvec_rows(sys_, mu, rows) -> np.ndarray:
    n = sys_.n_atoms
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    mu = _f64(mu).reshape(n, 3)
    out = np.zeros((rows.size, 3))
    pos, al = _f64(sys_.pos), _f64(sys_.polarizability)
    lib().oracle_tmatvec_rows(n, _p(pos), _p(al), _p(mu), sys_.box, sys_.cutoff,
                              sys_.ewald_beta, sys_.thole_a, rows.size,
                              _p(rows, _i64p), _p(out))
    return out


def dense_T(sys_) -> np.ndarray:
    """Dense (3N,3N) T_real + self (small N only)."""
    n = sys_.n_atoms
    T = np.zeros((3 * n, 3 * n))
    pos, al = _f64(sys_.pos), _f64(sys_.polarizability)
    lib().oracle_dense_T(n, _p(pos), _p(al), sys_.box, sys_.cutoff, sys_.ewald_beta,
                         sys_.thole_a, _p(T))
    return T


def dense_A(sys_) -> np.ndarray:
    """(S) A = alpha^-1 - T  (BASELINE.json: "the solve operator is alpha^-1 minus
    the real-space T with the Ewald self term")."""
    inv_alpha = np.repeat(1.0 / _f64(sys_.polarizability), 3)
    return np.diag(inv_alpha) - dense_T(sys_)


def count_pairs(sys_) -> int:
    pos = _f64(sys_.pos)
    return int(lib().oracle_count_pairs(sys_.n_atoms, _p(pos), sys_.box, sys_.cutoff))


def count_pairs_rows(sys_, rows) -> int:
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    pos = _f64(sys_.pos)
    return int(lib().oracle_count_pairs_rows(sys_.n_atoms, _p(pos), sys_.box, sys_.cutoff,
                                             rows.size, _p(rows, _i64p)))


# ------------------------------------------------------------------ S, U
def pcg_solve(sys_, E, tol: float = 1e-6, max_iter: int = 100, guess=None):
    """(S) Jacobi-preconditioned CG on A mu = E, A mu = mu/alpha - T mu.

    Order of operations exactly as SURVEY 8(c) "S" / Q10:
    mu0 = alpha E (direct-field guess) unless a guess is given; r = E - A mu;
    z = alpha r; p = z; loop: q = A p; gamma = (r.z)/(p.q); mu += gamma p;
    r -= gamma q; test rms = sqrt(sum_i |r_i|^2 / N) < tol; z = alpha r;
    delta = (r.z)_new/(r.z)_old; p = z + delta p.
    Returns (mu, iterations, rms).  iterations = number of A p products in the loop.
    """
    n = sys_.n_atoms
    alpha = _f64(sys_.polarizability)[:, None]
    E = _f64(E).reshape(n, 3)

    def A(v):
        return v / alpha - tmatvec(sys_, v)

    mu = alpha * E if guess is None else _f64(guess).reshape(n, 3).copy()
    r = E - A(mu)
    z = alpha * r
    p = z.copy()
    rz = float(np.sum(r * z))
    rms = float(np.sqrt(np.sum(r * r) / n))
    it = 0
    while rms >= tol and it < max_iter:
        q = A(p)
        gamma = rz / float(np.sum(p * q))
        mu = mu + gamma * p
        r = r - gamma * q
        it += 1
        rms = float(np.sqrt(np.sum(r * r) / n))
        if rms < tol:
            break
        z = alpha * r
        rz_new = float(np.sum(r * z))
        delta = rz_new / rz
        rz = rz_new
        p = z + delta * p
    return mu, it, rms


def dense_solve(sys_, E) -> np.ndarray:
    """Reference mu for small N: dense A by Cholesky."""
    import scipy.linalg as sla
    n = sys_.n_atoms
    A = dense_A(sys_)
    c = sla.cho_factor(A, lower=True, check_finite=True)
    return sla.cho_solve(c, _f64(E).reshape(3 * n)).reshape(n, 3)


def polar_energy(mu, E) -> float:
    """(U) E_pol = -1/2 f sum_i mu_i . E_i, f = 332.063713 kcal A / (mol e^2)."""
    return float(-0.5 * COULOMB * np.sum(_f64(mu) * _f64(E)))


# ------------------------------------------------------------------ fixed point (paper eqs 2-3)
FIX_VEC_BITS = 34       # P:L287 "a 34 fractional bits has been selected for forces accumulation"
FIX_ENERGY_BITS = 30    # P:L287 "For the energy, we only allocated 30 fractional bits"


def to_fixed(x, frac_bits: int) -> np.ndarray:
    """Paper eq. (2): a = int(round(x * 2^fB)); round = to the nearest integer (ties to even)."""
    return np.rint(np.asarray(x, dtype=np.float64) * float(1 << frac_bits)).astype(np.int64)


def from_fixed(a, frac_bits: int) -> np.ndarray:
    """Paper eq. (3): x = real(a) / 2^fB."""
    return np.asarray(a, dtype=np.int64).astype(np.float64) / float(1 << frac_bits)


def polar_energy_fixed(mu, E) -> float:
    """Paper's FP mode for the energy (Q21): every ATOM's term
    -1/2 f mu_i . E_i is converted with eq. (2) at 30 fractional bits, the int64 terms are summed
    (exactly, in any order) and the sum is converted back with eq. (3).  The dot product is
    ((mu_x E_x + mu_y E_y) + mu_z E_z) in FP64 without fused multiply-adds, then times -f/2."""
    mu, E = _f64(mu), _f64(E)
    dot = (mu[:, 0] * E[:, 0] + mu[:, 1] * E[:, 1]) + mu[:, 2] * E[:, 2]
    terms = to_fixed(dot * (-0.5 * COULOMB), FIX_ENERGY_BITS)
    return float(from_fixed(int(terms.sum()), FIX_ENERGY_BITS))


# ------------------------------------------------------------------ N
def wrap(x: np.ndarray, box: float) -> np.ndarray:
    """(Q16) w = x - L floor(x/L), clamped into [0, L); identity when box <= 0."""
    x = _f64(x)
    if box <= 0:
        return x.copy()
    w = x - box * np.floor(x / box)
    w = np.where(w >= box, w - box, w)
    return np.where(w < 0.0, 0.0, w)


def grid_bits(extent: float) -> int:
    """smallest b in 1..8 with extent / 2^b <= 2.5 A (else 8)."""
    b = 1
    while extent / (1 << b) > 2.5 and b < 8:
        b += 1
    return b


OPEN_MAX_BITS = 6     # DESIGN.md "Sort key" (Q14): an open-boundary grid has at most 2^6 cells per axis


def cell_coords(pos: np.ndarray, box: float):
    """integer cell coordinates on a 2^b grid.

    periodic: w = wrap(x), extent = L, origin 0.  open boundary: origin = per-axis
    minimum, extent = 1.000001 * max_axis(max - min) + 1e-9, b <= 6 (wider systems get
    coarser cells: the order stays a deterministic function of the coordinates).
    cell = min(2^b - 1, floor(w * inv_h)), inv_h = 2^b / extent.
    Returns (cells (N,3) int64, b).
    """
    pos = _f64(pos)
    if box > 0:
        w = wrap(pos, box)
        extent = float(box)
    else:
        lo = pos.min(axis=0)
        w = pos - lo[None, :]
        extent = float((pos.max(axis=0) - lo).max()) * 1.000001 + 1e-9
    b = grid_bits(extent)
    if box <= 0:
        b = min(b, OPEN_MAX_BITS)
    inv_h = float(1 << b) / extent
    cells = np.floor(w * inv_h).astype(np.int64)
    cells = np.minimum(cells, (1 << b) - 1)
    cells = np.maximum(cells, 0)
    return cells, b


def hilbert_key(cells: np.ndarray, b: int) -> np.ndarray:
    """3-D Hilbert index of integer cell coordinates (Skilling 2004, "Programming
    the Hilbert curve": axes -> transposed index, then bit interleave, x first).
    Restated from the published algorithm; pinned by bijectivity and unit-step
    adjacency on full grids (tests/test_oracle_nblist.py)."""
    X = [np.array(cells[:, k], dtype=np.int64).copy() for k in range(3)]
    M = 1 << (b - 1)
    Q = M
    while Q > 1:
        P = Q - 1
        for i in range(3):
            hit = (X[i] & Q) != 0
            X[0] = np.where(hit, X[0] ^ P, X[0])
            t = np.where(hit, 0, (X[0] ^ X[i]) & P)
            X[0] ^= t
            X[i] ^= t
        Q >>= 1
    for i in range(1, 3):
        X[i] ^= X[i - 1]
    t = np.zeros_like(X[0])
    Q = M
    while Q > 1:
        t = np.where((X[2] & Q) != 0, t ^ (Q - 1), t)
        Q >>= 1
    for i in range(3):
        X[i] ^= t
    key = np.zeros_like(X[0])
    for k in range(b - 1, -1, -1):
        for i in range(3):
            key = (key << 1) | ((X[i] >> k) & 1)
    return key


def sort_keys(pos: np.ndarray, box: float) -> np.ndarray:
    cells, b = cell_coords(pos, box)
    return hilbert_key(cells, b)


def check_perm(perm: np.ndarray, pos: np.ndarray, box: float) -> None:
    """(N i,ii) perm is a permutation of 0..N-1 padded with -1 to 32*n_b, pads only
    at the end of the last block; order non-decreasing in (key, index)."""
    n = pos.shape[0]
    perm = np.asarray(perm)
    n_b = (n + 31) // 32
    assert perm.shape == (32 * n_b,), (perm.shape, n_b)
    real = perm[:n]
    assert np.all(perm[n:] == -1), "phantoms must fill the tail of the last block"
    assert np.array_equal(np.sort(real), np.arange(n)), "not a permutation"
    keys = sort_keys(pos, box)[real]
    dk = np.diff(keys)
    assert np.all(dk >= 0), "sort keys decrease along perm"
    ties = dk == 0
    assert np.all(np.diff(real)[ties] > 0), "ties must be ordered by original index"


def block_boxes(perm: np.ndarray, pos: np.ndarray, box: float):
    """(N iii)/(Q16) per-block centre and half-extent of the wrapped real atoms."""
    perm = np.ascontiguousarray(perm, dtype=np.int32)
    n_b = perm.size // 32
    pos = _f64(pos)
    c = np.zeros((n_b, 3))
    h = np.zeros((n_b, 3))
    lib().oracle_block_boxes(n_b, _p(perm, _i32p), _p(pos), box, _p(c), _p(h))
    return c, h


def block_pairs(perm: np.ndarray, pos: np.ndarray, box: float, reach: float) -> np.ndarray:
    """(N iii) brute-force set {(I,J): I <= J, box gap^2 <= reach^2}, (T,2) int32,
    lexicographic.  ``reach`` = cutoff + skin; reach^2 is formed once here."""
    c, h = block_boxes(perm, pos, box)
    n_b = c.shape[0]
    reach2 = float(reach) * float(reach)
    total = lib().oracle_block_pairs(n_b, _p(c), _p(h), box, reach2, None, 0)
    pairs = np.zeros((total, 2), dtype=np.int32)
    got = lib().oracle_block_pairs(n_b, _p(c), _p(h), box, reach2, _p(pairs, _i32p), total)
    assert got == total
    return pairs


def atom_pairs_covered(perm, pairs, pos, box, reach) -> bool:
    """(N iv) safety: every atom pair with R <= reach has its block pair listed
    (atom-level brute force, small/medium N)."""
    perm = np.asarray(perm)
    n = pos.shape[0]
    blk_of = np.empty(n, dtype=np.int64)
    real = perm >= 0
    blk_of[perm[real]] = np.nonzero(real)[0] // 32
    n_b = perm.size // 32
    listed = set((int(a) * n_b + int(b)) for a, b in np.asarray(pairs))
    pos = _f64(pos)
    r2 = reach * reach
    for i in range(n):
        d = pos[i][None, :] - pos[i + 1:]
        if box > 0:
            d -= box * np.round(d / box)
        close = np.nonzero(np.einsum("ij,ij->i", d, d) <= r2)[0] + i + 1
        bi = blk_of[i]
        for bj in np.unique(blk_of[close]):
            a, b = (bi, bj) if bi <= bj else (bj, bi)
            if int(a) * n_b + int(b) not in listed:
                return False
    return True
