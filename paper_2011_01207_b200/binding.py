"""ctypes binding of libtkhp.so -- same names as include/tkhp.h, marshalling only."""
from __future__ import annotations

import ctypes
from ctypes import (POINTER, Structure, byref, c_char_p, c_double, c_int32, c_int64,
                    c_size_t, c_void_p)
from pathlib import Path

TKHP_OK = 0
TKHP_EINVAL, TKHP_ECUDA, TKHP_ECUTOFF, TKHP_ENOLIST = -1, -2, -3, -4
TKHP_ENOCONV, TKHP_ECAPACITY, TKHP_ENONFINITE = -5, -6, -7
TKHP_FP64, TKHP_MIXED, TKHP_FIXED = 0, 1, 2
TKHP_LIST_TILES, TKHP_LIST_CLUSTER, TKHP_LIST_ATOM = 0, 1, 2
TKHP_SOLVER_NO_PERSISTENT, TKHP_SOLVER_NO_FUSED_STEP, TKHP_SOLVER_STORED_T = 1, 2, 4
TKHP_SOLVER_TEST_BARRIER_FAULT = 8
TKHP_STATIC_MAX_ATOMS = 4194304

_ERR_NAMES = {-1: "TKHP_EINVAL", -2: "TKHP_ECUDA", -3: "TKHP_ECUTOFF", -4: "TKHP_ENOLIST",
              -5: "TKHP_ENOCONV", -6: "TKHP_ECAPACITY", -7: "TKHP_ENONFINITE"}

EXPORTED_SYMBOLS = [
    "tkhp_workspace_bytes", "tkhp_create", "tkhp_destroy", "tkhp_last_error",
    "tkhp_nblist_build", "tkhp_nblist_view", "tkhp_nblist_stats", "tkhp_nblist_atom_stats", "tkhp_perm_field",
    "tkhp_tmatvec", "tkhp_polar_solve", "tkhp_polar_energy", "tkhp_polar_energy_static", "tkhp_polarize_host",
    "tkhp_last_timings", "tkhp_fma_peak", "tkhp_profile_reset", "tkhp_profile_read",
    "tkhp_profile_read_solve", "tkhp_profile_read_build",
]


class TkhpError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"{_ERR_NAMES.get(code, code)}: {message}")
        self.code = code


class TkhpParams(Structure):
    """Mirror of ``tkhp_params``."""
    _fields_ = [("n_atoms", c_int32), ("precision", c_int32), ("device", c_int32),
                ("list_mode", c_int32), ("box", c_double), ("cutoff", c_double),
                ("skin", c_double), ("ewald_beta", c_double), ("thole_a", c_double),
                ("max_tiles_per_block", c_int32), ("max_nbrs_per_cluster", c_int32),
                ("max_nbrs_per_atom", c_int32), ("max_stage_per_chunk", c_int32),
                ("solver_flags", c_int32), ("reserved", c_int32)]


def lib_path() -> Path:
    return Path(__file__).resolve().parent / "libtkhp.so"


_lib = None


def lib() -> ctypes.CDLL:
    """Load libtkhp.so; raise loudly if the CUDA extension has not been built."""
    global _lib
    if _lib is None:
        path = lib_path()
        if not path.exists():
            raise ImportError(
                f"{path} is missing: build it with `python -m paper_2011_01207_b200.build` "
                "(nvcc, sm_100a). There is no CPU fallback.")
        L = ctypes.CDLL(str(path))
        vp, dp, ip = c_void_p, c_void_p, c_void_p   # device pointers travel as integers
        L.tkhp_workspace_bytes.argtypes = [POINTER(TkhpParams), POINTER(c_size_t)]
        L.tkhp_create.argtypes = [POINTER(TkhpParams), vp, c_size_t, POINTER(c_void_p)]
        L.tkhp_destroy.argtypes = [c_void_p]
        L.tkhp_last_error.argtypes = [c_void_p]
        L.tkhp_last_error.restype = c_char_p
        L.tkhp_nblist_build.argtypes = [c_void_p, dp, dp, ip, vp]
        L.tkhp_nblist_view.argtypes = [c_void_p, POINTER(c_int32), POINTER(c_int64),
                                       POINTER(c_void_p), POINTER(c_void_p), vp]
        L.tkhp_nblist_stats.argtypes = [c_void_p, POINTER(c_int64), POINTER(c_int64),
                                        POINTER(c_int32), vp]
        L.tkhp_nblist_atom_stats.argtypes = [c_void_p, POINTER(c_int64), vp]
        L.tkhp_perm_field.argtypes = [c_void_p, dp, dp, dp, dp, vp]
        L.tkhp_tmatvec.argtypes = [c_void_p, dp, dp, vp]
        L.tkhp_polar_solve.argtypes = [c_void_p, dp, dp, c_double, c_int32, c_int32,
                                       POINTER(c_int32), POINTER(c_double), vp]
        L.tkhp_polar_energy.argtypes = [c_void_p, dp, dp, dp, vp]
        L.tkhp_polar_energy_static.argtypes = [c_int32, c_int64, dp, dp, dp, vp]
        L.tkhp_polarize_host.argtypes = [c_void_p, vp, vp, vp, vp, vp, vp, c_double, c_int32,
                                         vp, vp, vp, POINTER(c_int32), POINTER(c_double), vp]
        L.tkhp_last_timings.argtypes = [c_void_p, POINTER(c_double)]
        L.tkhp_fma_peak.argtypes = [c_int32, c_int32, c_double, POINTER(c_double)]
        L.tkhp_profile_reset.argtypes = [c_void_p, c_int32]
        L.tkhp_profile_read.argtypes = [c_void_p, POINTER(c_int64), POINTER(c_int32),
                                        POINTER(c_double), POINTER(c_int32), POINTER(c_double)]
        L.tkhp_profile_read_solve.argtypes = [c_void_p, POINTER(c_int32), POINTER(c_double), POINTER(c_int64)]
        L.tkhp_profile_read_build.argtypes = [c_void_p, POINTER(c_int64)]
        for name in EXPORTED_SYMBOLS:
            if name != "tkhp_last_error":
                getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


def _check(rc: int, ctx=None, ok=(TKHP_OK,)):
    if rc not in ok:
        msg = lib().tkhp_last_error(ctx)
        raise TkhpError(rc, msg.decode() if msg else "")
    return rc


def _ptr(t):
    """Device pointer of a torch tensor (or a raw integer / None)."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return t.data_ptr()


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


# ---------------------------------------------------------------- 1:1 wrappers
def tkhp_workspace_bytes(params: TkhpParams) -> int:
    out = c_size_t(0)
    _check(lib().tkhp_workspace_bytes(byref(params), byref(out)))
    return out.value


def tkhp_create(params: TkhpParams, d_workspace, nbytes: int):
    ctx = c_void_p(None)
    _check(lib().tkhp_create(byref(params), _ptr(d_workspace), nbytes, byref(ctx)))
    return ctx


def tkhp_destroy(ctx):
    _check(lib().tkhp_destroy(ctx))


def tkhp_last_error(ctx=None) -> str:
    msg = lib().tkhp_last_error(ctx)
    return msg.decode() if msg else ""


def tkhp_nblist_build(ctx, d_pos, d_polarizability, d_group_id, stream=None):
    _check(lib().tkhp_nblist_build(ctx, _ptr(d_pos), _ptr(d_polarizability), _ptr(d_group_id),
                                   _stream_ptr(stream)), ctx)


def tkhp_nblist_view(ctx, stream=None):
    """-> (n_blocks, n_pairs, d_perm pointer, d_pairs pointer)."""
    nb, npairs = c_int32(0), c_int64(0)
    perm, pairs = c_void_p(None), c_void_p(None)
    _check(lib().tkhp_nblist_view(ctx, byref(nb), byref(npairs), byref(perm), byref(pairs),
                                  _stream_ptr(stream)), ctx)
    return nb.value, npairs.value, perm.value, pairs.value


def tkhp_nblist_stats(ctx, stream=None, count_pairs: bool = True):
    """-> (n_pairs_within_cutoff or None, n_slots_evaluated, list_mode_in_use)."""
    npair, nslot, mode = c_int64(-1), c_int64(0), c_int32(0)
    _check(lib().tkhp_nblist_stats(ctx, byref(npair) if count_pairs else None, byref(nslot),
                                   byref(mode), _stream_ptr(stream)), ctx)
    return (npair.value if count_pairs else None), nslot.value, mode.value


def tkhp_nblist_atom_stats(ctx, stream=None):
    """-> (far lane-slots, near lane-slots, segments, far class in use) of the ATOM lists."""
    out = (c_int64 * 4)()
    _check(lib().tkhp_nblist_atom_stats(ctx, out, _stream_ptr(stream)), ctx)
    return int(out[0]), int(out[1]), int(out[2]), bool(out[3])


def tkhp_perm_field(ctx, d_charge, d_dipole, d_quad, d_field, stream=None):
    _check(lib().tkhp_perm_field(ctx, _ptr(d_charge), _ptr(d_dipole), _ptr(d_quad), _ptr(d_field),
                                 _stream_ptr(stream)), ctx)


def tkhp_tmatvec(ctx, d_mu, d_out, stream=None):
    _check(lib().tkhp_tmatvec(ctx, _ptr(d_mu), _ptr(d_out), _stream_ptr(stream)), ctx)


def tkhp_polar_solve(ctx, d_field, d_mu, tol=1e-6, max_iter=100, use_guess=False, stream=None,
                     allow_noconv=False):
    """-> (iterations, rms, converged)."""
    it, rms = c_int32(0), c_double(0.0)
    ok = (TKHP_OK, TKHP_ENOCONV) if allow_noconv else (TKHP_OK,)
    rc = _check(lib().tkhp_polar_solve(ctx, _ptr(d_field), _ptr(d_mu), tol, max_iter,
                                       1 if use_guess else 0, byref(it), byref(rms),
                                       _stream_ptr(stream)), ctx, ok)
    return it.value, rms.value, rc == TKHP_OK


def tkhp_polar_energy(ctx, d_mu, d_field, d_energy, stream=None):
    _check(lib().tkhp_polar_energy(ctx, _ptr(d_mu), _ptr(d_field), _ptr(d_energy),
                                   _stream_ptr(stream)), ctx)


def tkhp_polar_energy_static(device: int, n_atoms: int, d_mu, d_field, d_energy, stream=None):
    """E_pol into ``d_energy`` without a context or a workspace, for code that may not allocate
    device memory (a plug-in inside an MD engine's step loop whose memory all belongs to the
    engine's pool, a callback running while a stream capture is open elsewhere, a loop that
    cannot take cudaMalloc's device-wide stall).  The reduction's scratch is a fixed 8,448-byte
    array inside libtkhp's device image; ``n_atoms`` may be at most ``TKHP_STATIC_MAX_ATOMS``.
    Calls on one GPU share that array: do not let two of them overlap.  See include/tkhp.h."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream(device)
    _check(lib().tkhp_polar_energy_static(device, n_atoms, _ptr(d_mu), _ptr(d_field), _ptr(d_energy),
                                          _stream_ptr(stream)))


def tkhp_polarize_host(ctx, h_pos, h_polarizability, h_group_id, h_charge, h_dipole, h_quad,
                       tol, max_iter, h_mu, h_field, h_energy, stream=None, allow_noconv=False):
    """Host-buffer entry; arguments are CPU tensors / numpy arrays (pinned preferred).
    -> (iterations, rms, converged)."""
    def hp(a):
        if a is None:
            return None
        if hasattr(a, "data_ptr"):
            return a.data_ptr()
        return a.ctypes.data
    it, rms = c_int32(0), c_double(0.0)
    ok = (TKHP_OK, TKHP_ENOCONV) if allow_noconv else (TKHP_OK,)
    rc = _check(lib().tkhp_polarize_host(ctx, hp(h_pos), hp(h_polarizability), hp(h_group_id),
                                         hp(h_charge), hp(h_dipole), hp(h_quad), tol, max_iter,
                                         hp(h_mu), hp(h_field), hp(h_energy), byref(it), byref(rms),
                                         _stream_ptr(stream)), ctx, ok)
    return it.value, rms.value, rc == TKHP_OK


def tkhp_last_timings(ctx):
    """-> dict of phase -> ms (negative: not run)."""
    arr = (c_double * 5)()
    _check(lib().tkhp_last_timings(ctx, arr), ctx)
    return dict(zip(("build", "field", "tmatvec", "solve", "energy"), list(arr)))


def tkhp_profile_reset(ctx, enable_kernel_events: bool = True):
    _check(lib().tkhp_profile_reset(ctx, 1 if enable_kernel_events else 0), ctx)


def tkhp_profile_read(ctx):
    """-> dict(launches, n_tmatvec, tmatvec_ms, n_field, field_ms)."""
    nl, nt, nf = c_int64(0), c_int32(0), c_int32(0)
    tt, tf = c_double(0.0), c_double(0.0)
    _check(lib().tkhp_profile_read(ctx, byref(nl), byref(nt), byref(tt), byref(nf), byref(tf)), ctx)
    return dict(launches=nl.value, n_tmatvec=nt.value, tmatvec_ms=tt.value, n_field=nf.value,
                field_ms=tf.value)


def tkhp_profile_read_solve(ctx):
    """-> dict(n_solve, solve_ms, solve_matvecs) of the persistent PCG kernel."""
    n, ms, mv = c_int32(0), c_double(0.0), c_int64(0)
    _check(lib().tkhp_profile_read_solve(ctx, byref(n), byref(ms), byref(mv)), ctx)
    return dict(n_solve=n.value, solve_ms=ms.value, solve_matvecs=mv.value)


def tkhp_profile_read_build(ctx):
    """-> dict(graph_captures, graph_replays, plain_builds, graphs_off) of this context's list builds,
    plus barrier_timeouts (persistent solves repeated on the launch-per-matvec path)."""
    out = (c_int64 * 5)()
    _check(lib().tkhp_profile_read_build(ctx, out), ctx)
    return dict(graph_captures=int(out[0]), graph_replays=int(out[1]), plain_builds=int(out[2]),
                graphs_off=bool(out[3]), barrier_timeouts=int(out[4]))


def tkhp_fma_peak(device: int, precision: int, seconds: float = 2.0) -> float:
    out = c_double(0.0)
    _check(lib().tkhp_fma_peak(device, precision, seconds, byref(out)))
    return out.value


# ---------------------------------------------------------------- convenience
class Polarizer:
    """Owns a workspace tensor and a context; methods mirror the C entry points.

    All array arguments are CUDA float64 / int32 torch tensors in original atom
    order; outputs are allocated by the caller or by the method (torch.empty).
    """

    def __init__(self, n_atoms, box, cutoff=7.0, skin=2.0, ewald_beta=0.5446, thole_a=0.39,
                 precision=TKHP_MIXED, list_mode=TKHP_LIST_TILES, device=0,
                 max_tiles_per_block=0, max_nbrs_per_cluster=0, max_nbrs_per_atom=0,
                 max_stage_per_chunk=0, solver_flags=0):
        import torch
        if not torch.cuda.is_available():
            raise TkhpError(TKHP_ECUDA, "no CUDA device: libtkhp has no CPU fallback")
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.params = TkhpParams(n_atoms, precision, device, list_mode, box, cutoff, skin,
                                 ewald_beta, thole_a, max_tiles_per_block, max_nbrs_per_cluster,
                                 max_nbrs_per_atom, max_stage_per_chunk, solver_flags, 0)
        self.n = n_atoms
        nbytes = tkhp_workspace_bytes(self.params)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) & ~255
            self.ctx = tkhp_create(self.params, self._ws_ptr, nbytes)
        self.workspace_bytes = nbytes

    @classmethod
    def for_system(cls, sys_, **kw):
        return cls(sys_.n_atoms, sys_.box, cutoff=sys_.cutoff, skin=sys_.skin,
                   ewald_beta=sys_.ewald_beta, thole_a=sys_.thole_a, **kw)

    def close(self):
        if getattr(self, "ctx", None) is not None:
            tkhp_destroy(self.ctx)
            self.ctx = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _s(self, stream):
        """The caller's stream, else the current stream of THIS context's device."""
        return self.torch.cuda.current_stream(self.device) if stream is None else stream

    def _f64(self, a):
        return self.torch.as_tensor(a, dtype=self.torch.float64, device=self.device).contiguous()

    # --- the five calls of the hot path
    def nblist_build(self, pos, polarizability, group_id, stream=None):
        t = self.torch
        self._pos = self._f64(pos)
        self._alpha = self._f64(polarizability)
        self._group = t.as_tensor(group_id, dtype=t.int32, device=self.device).contiguous()
        tkhp_nblist_build(self.ctx, self._pos, self._alpha, self._group, self._s(stream))

    def nblist_view(self, stream=None):
        """-> (perm (32*n_blocks,) int32 CPU numpy, pairs (T,2) int32 CPU numpy)."""
        import numpy as np
        nb, npairs, p_perm, p_pairs = tkhp_nblist_view(self.ctx, self._s(stream))
        off_perm = p_perm - self._ws_ptr
        off_pairs = p_pairs - self._ws_ptr
        base = self._ws_ptr - self.workspace.data_ptr()
        ws = self.workspace
        perm = ws[base + off_perm: base + off_perm + 4 * 32 * nb].view(self.torch.int32)
        pairs = ws[base + off_pairs: base + off_pairs + 8 * npairs].view(self.torch.int32)
        return perm.cpu().numpy().copy(), pairs.cpu().numpy().reshape(-1, 2).copy()

    def nblist_stats(self, stream=None, count_pairs=True):
        return tkhp_nblist_stats(self.ctx, self._s(stream), count_pairs)

    def nblist_atom_stats(self, stream=None):
        return tkhp_nblist_atom_stats(self.ctx, self._s(stream))

    def perm_field(self, charge, dipole, quad, out=None, stream=None):
        q, d, th = self._f64(charge), self._f64(dipole), self._f64(quad)
        if out is None:
            out = self.torch.empty((self.n, 3), dtype=self.torch.float64, device=self.device)
        tkhp_perm_field(self.ctx, q, d, th, out, self._s(stream))
        return out

    def tmatvec(self, mu, out=None, stream=None):
        mu = self._f64(mu)
        if out is None:
            out = self.torch.empty((self.n, 3), dtype=self.torch.float64, device=self.device)
        tkhp_tmatvec(self.ctx, mu, out, self._s(stream))
        return out

    def polar_solve(self, field, tol=1e-6, max_iter=100, guess=None, stream=None,
                    allow_noconv=False):
        """-> (mu, iterations, rms)."""
        field = self._f64(field)
        if guess is None:
            mu = self.torch.empty((self.n, 3), dtype=self.torch.float64, device=self.device)
        else:
            mu = self._f64(guess).clone()
        it, rms, _ = tkhp_polar_solve(self.ctx, field, mu, tol, max_iter, guess is not None, self._s(stream),
                                      allow_noconv)
        return mu, it, rms

    def polar_energy(self, mu, field, stream=None):
        """-> 0-d CUDA float64 tensor (kcal/mol)."""
        out = self.torch.empty((), dtype=self.torch.float64, device=self.device)
        tkhp_polar_energy(self.ctx, self._f64(mu), self._f64(field), out, self._s(stream))
        return out

    def timings(self):
        return tkhp_last_timings(self.ctx)
