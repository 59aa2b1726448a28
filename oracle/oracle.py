"""Python face of the CPU oracle (see pce_oracle.c for the header and the pins).

TEST INFRASTRUCTURE ONLY.  Plain numpy + ctypes; every function cites the
passage of /root/reference/PAPER.md (PAPER.md:line) it follows.  Conventions:
positions are (N, 3) float64 arrays, beads of body 0, 1, ... contiguous, ions
last; ``body_offset`` has N_body + 1 entries; eps_f defaults to 1 (the paper's
dimensionless units).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pce_oracle.c")
_LIB = os.path.join(_HERE, "liborc.so")
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)


def build(force: bool = False) -> str:
    """Compile pce_oracle.c with gcc (-O2 -fopenmp, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=gnu11", "-o", _LIB, _SRC, "-lm"]
        )
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        for name, n in (("orc_M_free", 2), ("orc_R", 3), ("orc_R0", 2), ("orc_dR", 3)):
            f = getattr(lib, name)
            f.restype = ctypes.c_double
            f.argtypes = [ctypes.c_double] * n
        lib.orc_ewald_eval.restype = ctypes.c_int
        lib.orc_ewald_eval.argtypes = [
            ctypes.c_int, _dp, _dp, _dp, _dp, ctypes.c_int, _ip, _dp,
            ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int,
            _dp, _dp, _dp, _dp,
        ]
        lib.orc_pair_matrix.restype = ctypes.c_int
        lib.orc_pair_matrix.argtypes = [
            ctypes.c_int, _dp, _dp, _dp, _dp,
            ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double, _dp,
        ]
        lib.orc_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().orc_num_threads())


def _d(a):
    return a.ctypes.data_as(_dp)


# ---------------------------------------------------------------- kernels
def M_free(r, a, eps=1.0):
    """eq. 10, repaired per reading G1."""
    return _load().orc_M_free(float(r), float(a)) / eps


def R(r, a, xi, eps=1.0):
    """eq. 20, Heaviside sign per reading G3."""
    return _load().orc_R(float(r), float(a), float(xi)) / eps


def R0(a, xi, eps=1.0):
    """eq. 21."""
    return _load().orc_R0(float(a), float(xi)) / eps


def dR(r, a, xi, eps=1.0):
    """d/dr of eq. 20 (reading A2)."""
    return _load().orc_dR(float(r), float(a), float(xi)) / eps


def default_xi(L, s=6.0):
    """The oracle's own splitting parameter: s/xi_o = min(L)/2 (r_c,o = s/xi_o + 2a)."""
    return 2.0 * s / float(np.min(L))


# ---------------------------------------------------------------- operator
def ewald_eval(x, q, L, a, eps=1.0, xi=None, s=6.0, targets=None, field=True):
    """psi = M q (eq. 8) and E = -grad(M q) at ``targets``
    (indices into x; default all), by the direct Ewald sum of eq. 19
     with the oracle's own xi, r_c = s/xi + 2a, k_max = 2 s xi."""
    lib = _load()
    x = np.ascontiguousarray(x, dtype=np.float64)
    N = x.shape[0]
    xs, ys, zs = (np.ascontiguousarray(x[:, i]) for i in range(3))
    q = np.ascontiguousarray(q, dtype=np.float64)
    assert q.shape == (N,)
    L = np.ascontiguousarray(np.broadcast_to(np.asarray(L, dtype=np.float64), (3,)))
    if xi is None:
        xi = default_xi(L, s)
    if targets is None:
        targets = np.arange(N)
    t = np.ascontiguousarray(targets, dtype=np.int32)
    Nt = t.shape[0]
    psi = np.zeros(Nt)
    E = np.zeros((3, Nt))
    rc = lib.orc_ewald_eval(
        N, _d(xs), _d(ys), _d(zs), _d(q), Nt, t.ctypes.data_as(_ip), _d(L),
        float(a), float(eps), float(xi), float(s), int(bool(field)),
        _d(psi), _d(E[0]), _d(E[1]), _d(E[2]),
    )
    if rc != 0:
        raise ValueError("orc_ewald_eval: bad arguments")
    return (psi, E.T.copy()) if field else psi


def pair_matrix(x, L, a, eps=1.0, xi=None, s=6.0):
    """Dense potential tensor M (eq. 9) entry by entry.  Default
    xi puts r_c,o at 1.5 min(L): few wave vectors, ~14 images per pair."""
    lib = _load()
    x = np.ascontiguousarray(x, dtype=np.float64)
    N = x.shape[0]
    xs, ys, zs = (np.ascontiguousarray(x[:, i]) for i in range(3))
    L = np.ascontiguousarray(np.broadcast_to(np.asarray(L, dtype=np.float64), (3,)))
    if xi is None:
        xi = s / (1.5 * float(np.min(L)))
    M = np.zeros((N, N))
    rc = lib.orc_pair_matrix(N, _d(xs), _d(ys), _d(zs), _d(L), float(a), float(eps), float(xi), float(s), _d(M))
    if rc != 0:
        raise ValueError("orc_pair_matrix: bad arguments")
    return M


# ---------------------------------------------------------------- bodies
def body_centres(x, body_offset, L):
    """X_i = mean of the body's bead positions after unwrapping every bead to
    the image nearest the body's first bead ("centre of mass", PAPER.md:115;
    reading A7).  Returns (X (N_body,3), r (N_bead,3) = x_ij - X_i, eq. 12)."""
    x = np.asarray(x, dtype=np.float64)
    L = np.broadcast_to(np.asarray(L, dtype=np.float64), (3,))
    off = np.asarray(body_offset, dtype=np.int64)
    nb = len(off) - 1
    X = np.zeros((nb, 3))
    r = np.zeros((off[-1], 3))
    for i in range(nb):
        xb = x[off[i]:off[i + 1]]
        d = xb - xb[0]
        d -= L * np.round(d / L)
        X[i] = xb[0] + d.mean(axis=0)
        r[off[i]:off[i + 1]] = d - d.mean(axis=0)
    return X, r


def rel_positions(x, body_offset, L):
    return body_centres(x, body_offset, L)[1]


def _sigma_apply(v, off):
    """Sigma . v : per-body sums (rows of consecutive ones, eq. 52)."""
    return np.add.reduceat(v, off[:-1]) if len(off) > 1 else np.zeros(0)


def solve_induced(x, body_offset, Q_body, q_ion, E0, L, a, eps=1.0, method="dense",
                  xi=None, s=6.0, cg_tol=1e-13, cg_maxit=2000):
    """Induced bead charges and body potentials: eq. 13,
        [-M  Sigma^T; Sigma  0] [q; Phi] = [-r.E0; Q],   Phi_i = Psi_i - Psi_0,i ,
    with the ions (one-bead bodies of fixed charge) eliminated:
        M_bb q_b - Sigma_b^T Phi_b = r.E0 - M_bi q_i ,  Sigma_b q_b = Q_b .
    method="dense": dense M_bb (pair_matrix) + LAPACK LU of the KKT matrix.
    method="cg"   : CG on the per-body-mean-projected system with the direct
                    Ewald matvec (unique solution: M is SPD).
    Returns q (N, beads then ions), Phi_body (N_body), info dict."""
    x = np.asarray(x, dtype=np.float64)
    off = np.asarray(body_offset, dtype=np.int64)
    nb = len(off) - 1
    Nbead = int(off[-1])
    N = x.shape[0]
    q_ion = np.asarray(q_ion, dtype=np.float64)
    assert q_ion.shape == (N - Nbead,)
    Q_body = np.asarray(Q_body, dtype=np.float64)
    E0 = np.asarray(E0, dtype=np.float64)
    _, r = body_centres(x, off, L)
    rhs = r @ E0
    if N > Nbead:
        qi = np.concatenate([np.zeros(Nbead), q_ion])
        rhs = rhs - ewald_eval(x, qi, L, a, eps, xi=xi, s=s, targets=np.arange(Nbead), field=False)
    info = {"method": method}
    xb = x[:Nbead]
    if method == "dense":
        M = pair_matrix(xb, L, a, eps, s=s)
        K = np.zeros((Nbead + nb, Nbead + nb))
        K[:Nbead, :Nbead] = -M
        for i in range(nb):
            K[off[i]:off[i + 1], Nbead + i] = 1.0
            K[Nbead + i, off[i]:off[i + 1]] = 1.0
        sol = np.linalg.solve(K, np.concatenate([-rhs, Q_body]))
        qb, Phi = sol[:Nbead], sol[Nbead:]
        res = K @ sol - np.concatenate([-rhs, Q_body])
        info["kkt_residual"] = float(np.linalg.norm(res) / max(np.linalg.norm(rhs), 1e-300))
        info["M_bb"] = M
    elif method == "cg":
        cnt = np.diff(off).astype(np.float64)
        bid = np.repeat(np.arange(nb), np.diff(off))

        def proj(v):
            return v - (_sigma_apply(v, off) / cnt)[bid]

        def mv(v):
            return ewald_eval(xb, v, L, a, eps, xi=xi, s=s, field=False)

        qb = (Q_body / cnt)[bid]
        g = proj(rhs - mv(qb))
        p = g.copy()
        gg = g @ g
        g0 = np.sqrt(gg)
        it = 0
        while it < cg_maxit and np.sqrt(gg) > cg_tol * max(g0, 1e-300):
            Ap = proj(mv(p))
            al = gg / (p @ Ap)
            qb = qb + al * p
            g = g - al * Ap
            gn = g @ g
            p = g + (gn / gg) * p
            gg = gn
            it += 1
        Phi = _sigma_apply(mv(qb) - rhs, off) / cnt
        info["iters"] = it
        info["rel_resid"] = float(np.sqrt(gg) / max(g0, 1e-300))
    else:
        raise ValueError(method)
    return np.concatenate([qb, q_ion]), Phi, info


def forces_torques(x, body_offset, q, E0, L, a, eps=1.0, Phi_body=None, xi=None, s=6.0, targets=None):
    """Everything downstream of the solve:
      psi = M q, E = -grad(M q)                      (eq. 8 / eq. 19)
      f_a = q_a (E0 + E_a)                           (eq. 17 = eq. 58; the
            beta = alpha term of grad M vanishes, M symmetric)
      F_i = sum_j f_ij,  L_i = sum_j r_ij x f_ij     (eq. 18)
      S_i = sum_j r_ij q_ij                          (eq. 14)
      U_i = (Q_i Psi_i - S_i.E0)/2, Psi_i = Phi_i - X_i.E0   (eq. 16 line 1)
      U_MM = q.M.q/2;  W = U_MM - sum_a q_a x_a.E0   (reading A8).
    Returns a dict."""
    x = np.asarray(x, dtype=np.float64)
    off = np.asarray(body_offset, dtype=np.int64)
    nb = len(off) - 1
    Nbead = int(off[-1])
    N = x.shape[0]
    q = np.asarray(q, dtype=np.float64)
    E0 = np.asarray(E0, dtype=np.float64)
    psi, E = ewald_eval(x, q, L, a, eps, xi=xi, s=s, targets=targets, field=True)
    out = {"psi": psi, "E": E}
    if targets is not None:
        return out
    f = q[:, None] * (E0[None, :] + E)
    X, r = body_centres(x, off, L)
    F = np.zeros((nb, 3)); T = np.zeros((nb, 3)); S = np.zeros((nb, 3)); Qb = np.zeros(nb)
    for i in range(nb):
        sl = slice(off[i], off[i + 1])
        F[i] = f[sl].sum(axis=0)
        T[i] = np.cross(r[sl], f[sl]).sum(axis=0)
        S[i] = (r[sl] * q[sl, None]).sum(axis=0)
        Qb[i] = q[sl].sum()
    out.update(f=f, F=F, T=T, S=S, X=X, r=r)
    U_MM = 0.5 * float(q @ psi)
    xun = np.concatenate([np.repeat(X, np.diff(off), axis=0) + r, x[Nbead:]])
    W = U_MM - float(q @ (xun @ E0))
    out.update(U_MM=U_MM, W=W)
    if Phi_body is None:
        cnt = np.diff(off)
        Phi_body = np.array([(psi[off[i]:off[i + 1]] - r[off[i]:off[i + 1]] @ E0).mean() for i in range(nb)]) if nb else np.zeros(0)
    Psi_body = Phi_body - X @ E0
    U_body = 0.5 * (Qb * Psi_body - S @ E0)
    # ions: one-bead bodies, r = 0, S = 0, Phi_ion = (M q)_ion
    Psi_ion = psi[Nbead:] - x[Nbead:] @ E0
    U_ion = 0.5 * q[Nbead:] * Psi_ion
    out.update(U_body=np.concatenate([U_body, U_ion]), U_eq16=float(U_body.sum() + U_ion.sum()),
               Phi_body=Phi_body)
    return out


# ---------------------------------------------------------------- grand capacitance tensor (eq. 15) and eps_eff (eq. 36)
def sigma_prime(x, body_offset, L):
    """Sigma' (Appendix eq. 52-53): the 4 N_body x N_bead summation tensor whose first N_body rows are
    Sigma (consecutive ones over the beads of each body) and whose next 3 N_body rows carry r_ij in place of the ones;
    row N_body + 3 i + d holds component d of r_ij for body i."""
    off = np.asarray(body_offset, dtype=np.int64)
    nb, nbead = len(off) - 1, int(off[-1])
    _, r = body_centres(x, off, L)
    Sp = np.zeros((4 * nb, nbead))
    for i in range(nb):
        sl = slice(off[i], off[i + 1])
        Sp[i, sl] = 1.0
        for d in range(3):
            Sp[nb + 3 * i + d, sl] = r[sl, d]
    return Sp


def capacitance(x, body_offset, L, a, eps=1.0, s=6.0):
    """Grand capacitance tensor C = Sigma' M^-1 Sigma'^T (eq. 15) of the conductor bodies, dense:
    [Q; S] = C [Psi - Psi_0; E_0].  M is the bead-bead potential tensor (eq. 9) of the N_bead beads alone (ions are not
    conductors and carry no unknowns).  Returns the 4 N_body x 4 N_body matrix, blocks as in eq. 37:
    C[:nb, :nb] = C_qPsi, C[:nb, nb:] = C_qE, C[nb:, :nb] = C_SPsi, C[nb:, nb:] = C_SE."""
    off = np.asarray(body_offset, dtype=np.int64)
    nbead = int(off[-1])
    M = pair_matrix(np.asarray(x, dtype=np.float64)[:nbead], L, a, eps, s=s)
    Sp = sigma_prime(x, off, L)
    return Sp @ np.linalg.solve(M, Sp.T)


def effective_permittivity(C, n_body, V, eps=1.0):
    """eq. 36: eps_eff = eps_f - n <C_SPsi C_qPsi^-1 C_qE - C_SE>, n = N_body / V, with <.> the average over
    the bodies of the response to a field that is the same on every body: <X> = (1/N_b) sum_ij X_ij (3 x 3 blocks)."""
    nb = n_body
    Cq, CqE, CS, CSE = C[:nb, :nb], C[:nb, nb:], C[nb:, :nb], C[nb:, nb:]
    X = CS @ np.linalg.solve(Cq, CqE) - CSE          # (3 nb) x (3 nb)
    avg = X.reshape(nb, 3, nb, 3).sum(axis=(0, 2)) / nb
    return eps * np.eye(3) - (nb / V) * avg
