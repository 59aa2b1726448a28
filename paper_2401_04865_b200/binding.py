"""Thin ctypes binding of libpce.so (include/pce.h) -- argument marshalling only.

Every step of the hot path runs in the CUDA library; torch is used for device
memory and streams.  There is no CPU fallback: importing works anywhere (so
the symbol table can be checked), but creating a context without a CUDA
device, or without the built library, raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None

PCE_OK, PCE_EINVAL, PCE_ENOMEM, PCE_ECUDA, PCE_ECUFFT, PCE_ENOCONV, PCE_ESTATE = 0, -1, -2, -3, -4, -5, -6

EXPORTS = (
    "pce_suggest_params", "pce_create", "pce_destroy", "pce_last_error", "pce_set_system", "pce_set_positions",
    "pce_matvec", "pce_evaluate", "pce_solve", "pce_forces", "pce_step_host", "pce_set_timing", "pce_get_timings",
    "pce_get_info", "pce_launch_count", "pce_real_kernel_host", "pce_measure_fp64_peaks", "pce_debug_poison_shared_memory",
    "pce_capacitance_columns", "pce_effective_permittivity", "pce_bd_step", "pce_radial_profile", "pce_set_centres",
    "pce_radial_profile_static",
)


class PceParams(C.Structure):
    _fields_ = [("L", C.c_double * 3), ("Ng", C.c_int * 3), ("xi", C.c_double), ("rc", C.c_double), ("P", C.c_int),
                ("a", C.c_double), ("eps_f", C.c_double), ("tol_solver", C.c_double), ("max_iter", C.c_int),
                ("flags", C.c_int), ("P_matvec", C.c_int)]


class PceSolveInfo(C.Structure):
    _fields_ = [("iters", C.c_int), ("matvecs", C.c_int), ("rel_resid", C.c_double), ("converged", C.c_int),
                ("graph_replays", C.c_int)]


class PceBdParams(C.Structure):
    _fields_ = [("dt", C.c_double), ("gamma", C.c_double), ("kT", C.c_double), ("seed", C.c_ulonglong), ("step", C.c_uint),
                ("move_bodies", C.c_int)]


class PceTimings(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("cells", "real", "spread", "fft", "scale", "ifft", "gather", "krylov", "other", "total")] + \
               [(n, C.c_double) for n in ("bead_real", "bead_spread", "bead_gather")] + \
               [("n_matvec_bead", C.c_int), ("n_eval_full", C.c_int), ("n_fft_pairs", C.c_int)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class PceInfo(C.Structure):
    _fields_ = [("eta", C.c_double * 3), ("h", C.c_double * 3), ("ncell", C.c_int * 3), ("image_range", C.c_int * 3),
                ("nnz_near", C.c_longlong), ("N", C.c_int), ("N_bead", C.c_int), ("N_body", C.c_int),
                ("bytes_workspace", C.c_longlong), ("bytes_precond", C.c_longlong), ("n_precond_blocks", C.c_int), ("P_matvec", C.c_int), ("fft_mode", C.c_int)]


class PceError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"pce error {code}: {msg}")
        self.code = code


def lib_path() -> str:
    return _build.LIB


def load():
    """dlopen libpce.so (must have been built in-tree: see build.py / __graft_entry__.build)."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise PceError(PCE_ESTATE, f"{path} not built; run `python -m paper_2401_04865_b200.build` (no CPU fallback)")
    lib = C.CDLL(path)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
    lib.pce_suggest_params.argtypes = [dp, ip, C.c_double, C.c_double, C.c_int, C.POINTER(PceParams)]
    lib.pce_create.argtypes = [C.POINTER(PceParams), vp, C.POINTER(vp)]
    lib.pce_destroy.argtypes = [vp]
    lib.pce_last_error.argtypes = [vp]
    lib.pce_last_error.restype = C.c_char_p
    lib.pce_set_system.argtypes = [vp, C.c_int, C.c_int, ip, vp, vp, vp]
    lib.pce_set_positions.argtypes = [vp, vp, vp, vp]
    lib.pce_set_centres.argtypes = [vp, vp, vp, vp]
    lib.pce_matvec.argtypes = [vp, vp, vp]
    lib.pce_evaluate.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.pce_solve.argtypes = [vp, vp, vp, dp, C.c_int, vp, vp, C.POINTER(PceSolveInfo)]
    lib.pce_forces.argtypes = [vp, vp, dp] + [vp] * 9
    lib.pce_step_host.argtypes = [vp, vp, vp, vp, vp, vp, dp, C.c_int] + [vp] * 9 + [C.POINTER(PceSolveInfo)]
    lib.pce_set_timing.argtypes = [vp, C.c_int]
    lib.pce_get_timings.argtypes = [vp, C.POINTER(PceTimings)]
    lib.pce_get_info.argtypes = [vp, C.POINTER(PceInfo)]
    lib.pce_launch_count.argtypes = [vp]
    lib.pce_launch_count.restype = C.c_longlong
    lib.pce_measure_fp64_peaks.argtypes = [C.POINTER(C.c_double)]
    lib.pce_debug_poison_shared_memory.argtypes = [vp]
    lib.pce_capacitance_columns.argtypes = [vp, C.c_int, ip, vp, C.POINTER(PceSolveInfo)]
    lib.pce_effective_permittivity.argtypes = [vp, dp, C.POINTER(PceSolveInfo)]
    lib.pce_bd_step.argtypes = [vp, C.POINTER(PceBdParams)] + [vp] * 7
    lib.pce_radial_profile.argtypes = [vp, C.c_int, vp, C.c_double, C.c_int] + [vp] * 4
    lib.pce_radial_profile_static.argtypes = [vp, C.c_int, vp, vp, vp, vp, C.c_int, vp, dp, dp, C.c_double, C.c_double, C.c_int] + [vp] * 4 + \
                                             [C.c_char_p, C.c_int]
    lib.pce_real_kernel_host.argtypes = [C.c_double] * 4 + [C.c_int, dp, dp, dp]
    for n in EXPORTS:
        if n not in ("pce_last_error", "pce_launch_count"):
            getattr(lib, n).restype = C.c_int
    _lib = lib
    return lib


def real_kernel_host(a, xi, rc, r, eps_f=1.0):
    """R(r), dR/dr of eq. 20 as the device evaluates them (host-only test hook; NaN outside [a/4, rc))."""
    lib = load()
    r = np.ascontiguousarray(r, dtype=np.float64)
    R, dR = np.empty_like(r), np.empty_like(r)
    dp = C.POINTER(C.c_double)
    rc_ = lib.pce_real_kernel_host(float(a), float(xi), float(rc), float(eps_f), r.size, r.ctypes.data_as(dp), R.ctypes.data_as(dp),
                                   dR.ctypes.data_as(dp))
    if rc_ != PCE_OK:
        raise PceError(rc_, "pce_real_kernel_host: bad arguments")
    return R, dR


def measure_fp64_peaks():
    """(DFMA TFLOP/s, fp64 mma TFLOP/s) measured on the current CUDA device."""
    out = (C.c_double * 2)()
    rc_ = load().pce_measure_fp64_peaks(out)
    if rc_ != PCE_OK:
        raise PceError(rc_, "pce_measure_fp64_peaks failed (needs a CUDA device)")
    return float(out[0]), float(out[1])


def poison_shared_memory():
    """Test hook: fill every SM's shared memory with NaN patterns on the current torch stream."""
    import torch
    rc_ = load().pce_debug_poison_shared_memory(C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc_ != PCE_OK:
        raise PceError(rc_, "pce_debug_poison_shared_memory failed")


def _d3(v):
    return (C.c_double * 3)(*[float(t) for t in np.broadcast_to(np.asarray(v, dtype=np.float64), (3,))])


def suggest_params(L, Ng, a, tol=1e-10, P=0) -> PceParams:
    """pce_suggest_params: xi, r_c, P from eqs. 23, 28, 32."""
    lib = load()
    p = PceParams()
    ng = (C.c_int * 3)(*[int(t) for t in np.broadcast_to(np.asarray(Ng), (3,))])
    rc = lib.pce_suggest_params(_d3(L), ng, float(a), float(tol), int(P), C.byref(p))
    if rc:
        raise PceError(rc, "pce_suggest_params: invalid arguments")
    return p


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


PROFILE_STATIC_MAX_BINS = 16384  # PCE_PROFILE_STATIC_MAX_BINS of include/pce.h


def radial_profile_static(x, y, z, q_ion, q_bead, centre, L, a, r_lo, n_bins, out=None):
    """pce_radial_profile_static: the observables of Context.radial_profile without a context and without any device-memory
    allocation inside the library (its shell counters live in a fixed array of the library image) -- for callers that may not
    cudaMalloc, e.g. an analysis hook inside a simulation engine that has handed all device memory to its own pool.
    x, y, z, q_ion: contiguous CUDA float64 tensors of the ions; q_bead: charges of the body's beads (or None);
    ``out``: dict of preallocated tensors counts[2 n], g[2 n], rho[n], Qcum[n] to write into (this wrapper makes them with
    torch if not given: that allocation is the caller's, through torch's pool, not the library's).  n_bins is limited to
    PROFILE_STATIC_MAX_BINS.  Work is enqueued on the current torch stream; calls that overlap on the GPU race on the shared
    counters."""
    import torch
    n = int(x.numel())
    for t in (x, y, z, q_ion):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n, "need contiguous cuda f64"
    nb = 0 if q_bead is None else int(q_bead.numel())
    if q_bead is not None:
        assert q_bead.is_cuda and q_bead.dtype == torch.float64 and q_bead.is_contiguous(), "need contiguous cuda f64"
    if out is None:
        m = max(int(n_bins), 0)
        out = {k: torch.empty(s, dtype=torch.float64, device=x.device) for k, s in (("counts", 2 * m), ("g", 2 * m), ("rho", m), ("Qcum", m))}
    err = C.create_string_buffer(512)
    rc = load().pce_radial_profile_static(C.c_void_p(torch.cuda.current_stream().cuda_stream), n, _ptr(x), _ptr(y), _ptr(z), _ptr(q_ion), nb,
                                          _ptr(q_bead), _d3(centre), _d3(L), float(a), float(r_lo), int(n_bins), _ptr(out.get("counts")),
                                          _ptr(out.get("g")), _ptr(out.get("rho")), _ptr(out.get("Qcum")), err, len(err))
    if rc:
        raise PceError(rc, err.value.decode())
    return out


class Context:
    """RAII wrapper of a pce_ctx.  All tensors are torch float64 CUDA tensors
    (SoA); results are returned as new tensors."""

    def __init__(self, params: PceParams, stream=None):
        import torch

        self.torch = torch
        self.lib = load()
        if not torch.cuda.is_available():
            raise PceError(PCE_ECUDA, "no CUDA device: the library has no CPU fallback")
        self.params = params
        self.stream = stream
        s = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
        h = C.c_void_p()
        rc = self.lib.pce_create(C.byref(params), s, C.byref(h))
        if rc:
            raise PceError(rc, self.lib.pce_last_error(None).decode())
        self.h = h
        self.N = self.N_bead = self.N_body = 0

    def close(self):
        if getattr(self, "h", None):
            self.lib.pce_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc, allow=()):
        if rc and rc not in allow:
            raise PceError(rc, self.lib.pce_last_error(self.h).decode())
        return rc

    def _new(self, n):
        return self.torch.empty(int(n), dtype=self.torch.float64, device="cuda")

    def _chk(self, t, n):
        assert t.is_cuda and t.dtype == self.torch.float64 and t.is_contiguous() and t.numel() == n, "need contiguous cuda f64"

    # ---- system
    def set_system(self, body_offset, x, y, z):
        off = np.ascontiguousarray(body_offset, dtype=np.int32)
        N = x.numel()
        for t in (x, y, z):
            self._chk(t, N)
        self._ck(self.lib.pce_set_system(self.h, N, len(off) - 1, off.ctypes.data_as(C.POINTER(C.c_int)), _ptr(x), _ptr(y), _ptr(z)))
        self.N, self.N_body, self.N_bead = N, len(off) - 1, int(off[-1])

    def set_positions(self, x, y, z):
        for t in (x, y, z):
            self._chk(t, self.N)
        self._ck(self.lib.pce_set_positions(self.h, _ptr(x), _ptr(y), _ptr(z)))

    def set_centres(self, X, Y, Z):
        for t in (X, Y, Z):
            self._chk(t, self.N_body)
        self._ck(self.lib.pce_set_centres(self.h, _ptr(X), _ptr(Y), _ptr(Z)))

    # ---- operator
    def matvec(self, q):
        self._chk(q, self.N_bead)
        psi = self._new(self.N_bead)
        self._ck(self.lib.pce_matvec(self.h, _ptr(q), _ptr(psi)))
        return psi

    def evaluate(self, q, field=True):
        self._chk(q, self.N)
        psi = self._new(self.N)
        E = [self._new(self.N) for _ in range(3)] if field else [None] * 3
        self._ck(self.lib.pce_evaluate(self.h, _ptr(q), _ptr(psi), _ptr(E[0]), _ptr(E[1]), _ptr(E[2])))
        return (psi, E[0], E[1], E[2]) if field else psi

    # ---- solve / forces
    def solve(self, Q_body, q_ion, E0, q0=None, allow_noconv=False):
        self._chk(Q_body, self.N_body)
        if self.N - self.N_bead:
            self._chk(q_ion, self.N - self.N_bead)
        q = self._new(self.N)
        warm = 0
        if q0 is not None:
            q[: self.N_bead].copy_(q0[: self.N_bead])
            warm = 1
        Phi = self._new(self.N_body)
        info = PceSolveInfo()
        self._ck(self.lib.pce_solve(self.h, _ptr(Q_body), _ptr(q_ion) if self.N - self.N_bead else None, _d3(E0), warm,
                                    _ptr(q), _ptr(Phi), C.byref(info)), allow=(PCE_ENOCONV,) if allow_noconv else ())
        return q, Phi, {"iters": info.iters, "matvecs": info.matvecs, "rel_resid": info.rel_resid, "converged": bool(info.converged),
                        "graph_replays": info.graph_replays}

    def forces(self, q, E0):
        self._chk(q, self.N)
        nb, ni = self.N_body, self.N - self.N_bead
        f = [self._new(self.N) for _ in range(3)]
        F, T, S = self._new(3 * nb), self._new(3 * nb), self._new(3 * nb)
        Ub, Ut, psi = self._new(nb + ni), self._new(3), self._new(self.N)
        self._ck(self.lib.pce_forces(self.h, _ptr(q), _d3(E0), _ptr(f[0]), _ptr(f[1]), _ptr(f[2]), _ptr(F), _ptr(T), _ptr(S),
                                     _ptr(Ub), _ptr(Ut), _ptr(psi)))
        return {"f": self.torch.stack(f, dim=1), "F": F.view(3, nb).T, "T": T.view(3, nb).T, "S": S.view(3, nb).T,
                "U_body": Ub, "U_eq16": Ut[0], "W": Ut[1], "U_MM": Ut[2], "psi": psi}

    def capacitance_columns(self, cols):
        """Columns of C = Sigma' M^-1 Sigma'^T (eq. 15): tensor [len(cols), 4 N_body]."""
        cols = np.ascontiguousarray(cols, dtype=np.int32)
        out = self._new(len(cols) * 4 * self.N_body)
        info = PceSolveInfo()
        self._ck(self.lib.pce_capacitance_columns(self.h, len(cols), cols.ctypes.data_as(C.POINTER(C.c_int)), _ptr(out), C.byref(info)))
        return out.view(len(cols), 4 * self.N_body), {"iters": info.iters, "matvecs": info.matvecs, "rel_resid": info.rel_resid,
                                                        "converged": bool(info.converged)}

    def effective_permittivity(self):
        """eps_eff (3 x 3 numpy array), eq. 36."""
        out = (C.c_double * 9)()
        info = PceSolveInfo()
        self._ck(self.lib.pce_effective_permittivity(self.h, out, C.byref(info)))
        return np.array(list(out)).reshape(3, 3), {"iters": info.iters, "matvecs": info.matvecs, "rel_resid": info.rel_resid,
                                                    "converged": bool(info.converged)}

    def bd_step(self, f, dt, gamma=1.0, kT=1.0, seed=0, step=0, move_bodies=False, noise=None):
        """One Brownian-dynamics step (eqs. 40-46, 62) from the context's positions; f: (N, 3) forces of forces().
        noise: optional (N_ion, 3) standard normals (else the library's Philox stream).  Returns the new x, y, z."""
        fx, fy, fz = (f[:, d].contiguous() for d in range(3))
        for t in (fx, fy, fz):
            self._chk(t, self.N)
        nz = None
        if noise is not None:
            nz = noise.T.contiguous().view(-1)
            self._chk(nz, 3 * (self.N - self.N_bead))
        bp = PceBdParams(float(dt), float(gamma), float(kT), int(seed), int(step), int(bool(move_bodies)))
        x, y, z = self._new(self.N), self._new(self.N), self._new(self.N)
        self._ck(self.lib.pce_bd_step(self.h, C.byref(bp), _ptr(fx), _ptr(fy), _ptr(fz), _ptr(nz), _ptr(x), _ptr(y), _ptr(z)))
        return x, y, z

    def radial_profile(self, body, q, r_lo, n_bins):
        """Shell counts, g(r) (eq. 49), windowed charge density and Q'(r) (eq. 48) of the ions about a body's centre."""
        self._chk(q, self.N)
        counts, g, rho, Qc = self._new(2 * n_bins), self._new(2 * n_bins), self._new(n_bins), self._new(n_bins)
        self._ck(self.lib.pce_radial_profile(self.h, int(body), _ptr(q), float(r_lo), int(n_bins), _ptr(counts), _ptr(g), _ptr(rho), _ptr(Qc)))
        return {"counts": counts.view(2, n_bins).T, "g": g.view(2, n_bins).T, "rho": rho, "Qcum": Qc}

    def step_host(self, x, y, z, Q_body, q_ion, E0, out, warm_start=False):
        """Host-buffer pass.  x,y,z,Q_body,q_ion: host numpy/pinned-torch f64; ``out``: dict of host arrays
        (keys q, Phi, fx, fy, fz, F, T, S, U) written in place; warm_start: out["q"] holds the initial guess."""
        def hp(a):
            if a is None:
                return None
            return C.c_void_p(a.data_ptr()) if hasattr(a, "data_ptr") else C.c_void_p(a.ctypes.data)
        info = PceSolveInfo()
        rc = self._ck(self.lib.pce_step_host(self.h, hp(x), hp(y), hp(z), hp(Q_body), hp(q_ion), _d3(E0), int(bool(warm_start)), hp(out.get("q")),
                                             hp(out.get("Phi")), hp(out.get("fx")), hp(out.get("fy")), hp(out.get("fz")),
                                             hp(out.get("F")), hp(out.get("T")), hp(out.get("S")), hp(out.get("U")),
                                             C.byref(info)), allow=(PCE_ENOCONV,))
        return {"iters": info.iters, "matvecs": info.matvecs, "rel_resid": info.rel_resid, "converged": bool(info.converged), "rc": rc,
                "graph_replays": info.graph_replays}

    # ---- reports
    def set_timing(self, on=True):
        self._ck(self.lib.pce_set_timing(self.h, int(on)))

    def timings(self):
        t = PceTimings()
        self._ck(self.lib.pce_get_timings(self.h, C.byref(t)))
        return t.as_dict()

    def info(self):
        i = PceInfo()
        self._ck(self.lib.pce_get_info(self.h, C.byref(i)))
        return {"eta": list(i.eta), "h": list(i.h), "ncell": list(i.ncell), "image_range": list(i.image_range),
                "nnz_near": i.nnz_near, "N": i.N, "N_bead": i.N_bead, "N_body": i.N_body, "bytes_workspace": i.bytes_workspace,
                "bytes_precond": i.bytes_precond, "n_precond_blocks": i.n_precond_blocks, "P_matvec": i.P_matvec, "fft_mode": i.fft_mode}

    def launch_count(self):
        return int(self.lib.pce_launch_count(self.h))


PCE_FLAG_NO_PRECOND = 1
PCE_FLAG_CUFFT_3D = 2
PCE_FLAG_FIELD_IK = 4
PCE_FLAG_DETERMINISTIC = 8


def context_for(workload, tol=1e-10, P=0, tol_solver=1e-12, max_iter=500, stream=None, precond=True, fused_z=True, field_ik=False, deterministic=False, P_matvec=0) -> Context:
    """Context with parameters suggested for a workloads.Workload."""
    p = suggest_params(workload.L, workload.Ng, workload.a, tol, P)
    p.flags = (0 if precond else PCE_FLAG_NO_PRECOND) | (0 if fused_z else PCE_FLAG_CUFFT_3D) | (PCE_FLAG_FIELD_IK if field_ik else 0) | (PCE_FLAG_DETERMINISTIC if deterministic else 0)
    p.eps_f = workload.eps_f
    if P_matvec:
        p.P_matvec = int(P_matvec)
    p.tol_solver = tol_solver
    p.max_iter = max_iter
    return Context(p, stream)


def upload(workload):
    """Workload arrays as torch CUDA tensors: (x, y, z, Q_body, q_ion)."""
    import torch

    def t(a):
        return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    return t(workload.x[:, 0]), t(workload.x[:, 1]), t(workload.x[:, 2]), t(workload.Q_body), t(workload.q_ion)
