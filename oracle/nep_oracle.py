"""ctypes binding of oracle/nep_oracle.c (argument marshalling only).

TEST INFRASTRUCTURE: see the header of nep_oracle.c for what each routine states
and which passage of PAPER.md it follows."""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

__all__ = ["Hyper", "num_threads", "descriptor_dim", "num_params", "chebyshev", "cutoff", "radial",
           "legendre", "neighbors", "network", "descriptor_atom", "compute", "evaluate", "md", "md_driven",
           "loss", "snes_sample", "snes_utilities", "snes_update"]

_lib = C.CDLL(_build.build())
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


class Hyper(C.Structure):
    """Table I hyper-parameters; n_max inclusive (Eq. 16)."""
    _fields_ = [("rc_r", C.c_double), ("rc_a", C.c_double), ("nmax_r", C.c_int), ("nmax_a", C.c_int),
                ("lmax", C.c_int), ("nneu", C.c_int), ("ntypes", C.c_int),
                # variants (default 0 = the paper's own form): hidden layers 2-3 and the SOAP-like q_nn'l of Eq. 17
                ("nlayers", C.c_int), ("nneu2", C.c_int), ("nneu3", C.c_int), ("kind", C.c_int)]


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _i(a):
    return None if a is None else a.ctypes.data_as(_ip)


_lib.orc_num_threads.restype = C.c_int
_lib.orc_descriptor_dim.restype = C.c_int
_lib.orc_num_params.restype = C.c_int
for _f in ("orc_neighbors_brute", "orc_neighbors_cell", "orc_compute", "orc_evaluate", "orc_md", "orc_md_driven"):
    getattr(_lib, _f).restype = C.c_int


def num_threads() -> int:
    return _lib.orc_num_threads()


def descriptor_dim(h: Hyper) -> int:
    return _lib.orc_descriptor_dim(C.byref(h))


def num_params(h: Hyper) -> int:
    return _lib.orc_num_params(C.byref(h))


def chebyshev(x: float, nmax: int):
    T = np.zeros(nmax + 1); U = np.zeros(nmax + 1)
    _lib.orc_chebyshev(C.c_double(x), C.c_int(nmax), _d(T), _d(U))
    return T, U


def cutoff(r: float, rc: float):
    fc = C.c_double(); dfc = C.c_double()
    _lib.orc_cutoff(C.c_double(r), C.c_double(rc), C.byref(fc), C.byref(dfc))
    return fc.value, dfc.value


def radial(r: float, rc: float, nmax: int, omega: float = 1.0):
    g = np.zeros(nmax + 1); dg = np.zeros(nmax + 1)
    _lib.orc_radial(C.c_double(r), C.c_double(rc), C.c_int(nmax), C.c_double(omega), _d(g), _d(dg))
    return g, dg


def legendre(c: float, lmax: int):
    P = np.zeros(lmax + 1); dP = np.zeros(lmax + 1)
    _lib.orc_legendre(C.c_double(c), C.c_int(lmax), _d(P), _d(dP))
    return P, dP


def neighbors(pos, box, rc: float, cap: int, method: str = "brute"):
    """-> (count[N], index[N,cap] ascending rows, borderline pair count)."""
    pos = np.ascontiguousarray(pos, dtype=np.float64); box = np.ascontiguousarray(box, dtype=np.float64)
    n = pos.shape[1]
    count = np.zeros(n, dtype=np.int32); index = np.full((n, cap), -1, dtype=np.int32)
    nb = C.c_int64(0)
    fn = _lib.orc_neighbors_brute if method == "brute" else _lib.orc_neighbors_cell
    mx = fn(C.c_int64(n), _d(pos), _d(box), C.c_double(rc), C.c_int(cap), _i(count), _i(index), C.byref(nb))
    if mx > cap:
        raise OverflowError("neighbour capacity %d exceeded (max %d)" % (cap, mx))
    return count, index, nb.value


def network(h: Hyper, params, q):
    params = np.ascontiguousarray(params, dtype=np.float64); q = np.ascontiguousarray(q, dtype=np.float64)
    U = C.c_double(); Fp = np.zeros(descriptor_dim(h))
    _lib.orc_network(C.byref(h), _d(params), _d(q), C.byref(U), _d(Fp))
    return U.value, Fp


def descriptor_atom(h: Hyper, znum, types, pos, box, i, listR, listA):
    pos = np.ascontiguousarray(pos, dtype=np.float64); box = np.ascontiguousarray(box, dtype=np.float64)
    znum = np.ascontiguousarray(znum, dtype=np.int32); types = np.ascontiguousarray(types, dtype=np.int32)
    listR = np.ascontiguousarray(listR, dtype=np.int32); listA = np.ascontiguousarray(listA, dtype=np.int32)
    q = np.zeros(descriptor_dim(h))
    _lib.orc_descriptor_atom(C.byref(h), _i(znum), _i(types), C.c_int64(pos.shape[1]), _d(pos), _d(box),
                             C.c_int64(i), C.c_int(len(listR)), _i(listR), C.c_int(len(listA)), _i(listA), _d(q))
    return q


def compute(h: Hyper, znum, params, pos, vel, types, box, cntR, idxR, cntA, idxA, want_internals=False):
    """One evaluation with given lists -> dict(U, F[3,N], W[9,N], J[3,N] or None, [q, Fp, p])."""
    pos = np.ascontiguousarray(pos, dtype=np.float64); box = np.ascontiguousarray(box, dtype=np.float64)
    vel = None if vel is None else np.ascontiguousarray(vel, dtype=np.float64)
    znum = np.ascontiguousarray(znum, dtype=np.int32); types = np.ascontiguousarray(types, dtype=np.int32)
    params = np.ascontiguousarray(params, dtype=np.float64)
    assert params.size == num_params(h), (params.size, num_params(h))
    n = pos.shape[1]; D = descriptor_dim(h)
    capR, capA = idxR.shape[1], idxA.shape[1]
    out = dict(U=np.zeros(n), F=np.zeros((3, n)), W=np.zeros((9, n)), J=None if vel is None else np.zeros((3, n)))
    q = Fp = p = None
    if want_internals:
        q = np.zeros((n, D)); Fp = np.zeros((n, D)); p = np.zeros((n, capR, 3))
        out.update(q=q, Fp=Fp, p=p)
    rc = _lib.orc_compute(C.c_int64(n), _d(pos), _d(vel), _i(types), _d(box), C.byref(h), _i(znum), _d(params),
                          C.c_int(capR), _i(cntR), _i(idxR), C.c_int(capA), _i(cntA), _i(idxA),
                          _d(out["U"]), _d(out["F"]), _d(out["W"]), _d(out["J"]), _d(q), _d(Fp), _d(p))
    if rc:
        raise RuntimeError("orc_compute failed: %d" % rc)
    return out


def evaluate(h: Hyper, znum, params, pos, vel, types, box, capR=96, capA=64):
    """Lists from scratch (brute force for N<=8000, cell list above) + compute."""
    pos = np.ascontiguousarray(pos, dtype=np.float64); box = np.ascontiguousarray(box, dtype=np.float64)
    vel = None if vel is None else np.ascontiguousarray(vel, dtype=np.float64)
    znum = np.ascontiguousarray(znum, dtype=np.int32); types = np.ascontiguousarray(types, dtype=np.int32)
    params = np.ascontiguousarray(params, dtype=np.float64)
    assert params.size == num_params(h), (params.size, num_params(h))
    n = pos.shape[1]
    out = dict(U=np.zeros(n), F=np.zeros((3, n)), W=np.zeros((9, n)), J=None if vel is None else np.zeros((3, n)))
    rc = _lib.orc_evaluate(C.c_int64(n), _d(pos), _d(vel), _i(types), _d(box), C.byref(h), _i(znum), _d(params),
                           C.c_int(capR), C.c_int(capA), _d(out["U"]), _d(out["F"]), _d(out["W"]), _d(out["J"]))
    if rc:
        raise RuntimeError("orc_evaluate failed: %d" % rc)
    return out


def md(h: Hyper, znum, params, pos, vel, types, box, masses, dt, n_steps, capR=96, capA=64):
    """Velocity-Verlet NVE; returns dict(pos, vel, U, F, W, J, Jsum, thermo[n_steps+1,5])."""
    pos = np.array(pos, dtype=np.float64, order="C"); vel = np.array(vel, dtype=np.float64, order="C")
    box = np.ascontiguousarray(box, dtype=np.float64)
    znum = np.ascontiguousarray(znum, dtype=np.int32); types = np.ascontiguousarray(types, dtype=np.int32)
    params = np.ascontiguousarray(params, dtype=np.float64); masses = np.ascontiguousarray(masses, dtype=np.float64)
    n = pos.shape[1]
    out = dict(pos=pos, vel=vel, U=np.zeros(n), F=np.zeros((3, n)), W=np.zeros((9, n)), J=np.zeros((3, n)),
               Jsum=np.zeros((3, n)), thermo=np.zeros((n_steps + 1, 5)))
    rc = _lib.orc_md(C.c_int64(n), _d(pos), _d(vel), _i(types), _d(box), C.byref(h), _i(znum), _d(params),
                     _d(masses), C.c_double(dt), C.c_int(n_steps), C.c_int(capR), C.c_int(capA),
                     _d(out["U"]), _d(out["F"]), _d(out["W"]), _d(out["J"]), _d(out["Jsum"]), _d(out["thermo"]))
    if rc:
        raise RuntimeError("orc_md failed: %d" % rc)
    return out


def md_driven(h: Hyper, znum, params, pos, vel, types, box, masses, dt, n_steps, Fe=None, W0=None, capR=96, capA=64):
    """Velocity Verlet with the HNEMD driving force F_i += F_e . W_i (Eq. 9) and K(t) = sum_i W_i(0) . v_i(t)
    (Eq. 11); Fe=None is NVE.  Returns md()'s dict plus Kt[n_steps+1,3]."""
    pos = np.array(pos, dtype=np.float64, order="C"); vel = np.array(vel, dtype=np.float64, order="C")
    box = np.ascontiguousarray(box, dtype=np.float64)
    znum = np.ascontiguousarray(znum, dtype=np.int32); types = np.ascontiguousarray(types, dtype=np.int32)
    params = np.ascontiguousarray(params, dtype=np.float64); masses = np.ascontiguousarray(masses, dtype=np.float64)
    fe = None if Fe is None else np.ascontiguousarray(Fe, dtype=np.float64)
    w0 = None if W0 is None else np.ascontiguousarray(W0, dtype=np.float64)
    n = pos.shape[1]
    out = dict(pos=pos, vel=vel, U=np.zeros(n), F=np.zeros((3, n)), W=np.zeros((9, n)), J=np.zeros((3, n)),
               Jsum=np.zeros((3, n)), thermo=np.zeros((n_steps + 1, 5)), Kt=np.zeros((n_steps + 1, 3)))
    rc = _lib.orc_md_driven(C.c_int64(n), _d(pos), _d(vel), _i(types), _d(box), C.byref(h), _i(znum), _d(params),
                            _d(masses), C.c_double(dt), C.c_int(n_steps), C.c_int(capR), C.c_int(capA),
                            _d(fe), _d(w0), _d(out["Kt"]),
                            _d(out["U"]), _d(out["F"]), _d(out["W"]), _d(out["J"]), _d(out["Jsum"]), _d(out["thermo"]))
    if rc:
        raise RuntimeError("orc_md_driven failed: %d" % rc)
    return out


_lib.orc_loss.restype = C.c_int


def loss(h: Hyper, znum, z, first, pos, types, boxes, e_tar, f_tar, v_tar, lambdas, capR=96, capA=64):
    """Eq. 29-34 for one parameter vector: -> [L_e, L_f, L_v, L_1, L_2, L]."""
    first = np.ascontiguousarray(first, dtype=np.int64); pos = np.ascontiguousarray(pos, dtype=np.float64)
    types = np.ascontiguousarray(types, dtype=np.int32); boxes = np.ascontiguousarray(boxes, dtype=np.float64)
    znum = np.ascontiguousarray(znum, dtype=np.int32); z = np.ascontiguousarray(z, dtype=np.float64)
    e_tar = np.ascontiguousarray(e_tar, dtype=np.float64); f_tar = np.ascontiguousarray(f_tar, dtype=np.float64)
    v_tar = np.ascontiguousarray(v_tar, dtype=np.float64); lam = np.ascontiguousarray(lambdas, dtype=np.float64)
    assert z.size == num_params(h)
    out = np.zeros(6)
    rc = _lib.orc_loss(C.c_int(len(first) - 1), first.ctypes.data_as(C.POINTER(C.c_int64)), _d(pos), _i(types), _d(boxes),
                       C.byref(h), _i(znum), _d(z), C.c_int(capR), C.c_int(capA), _d(e_tar), _d(f_tar), _d(v_tar), _d(lam), _d(out))
    if rc:
        raise RuntimeError("orc_loss failed: %d" % rc)
    return out


def snes_sample(m, s, r):
    m = np.ascontiguousarray(m, dtype=np.float64); s = np.ascontiguousarray(s, dtype=np.float64)
    r = np.ascontiguousarray(r, dtype=np.float64)
    z = np.zeros_like(r)
    _lib.orc_snes_sample(C.c_int(r.shape[0]), C.c_int(r.shape[1]), _d(m), _d(s), _d(r), _d(z))
    return z


def snes_utilities(losses):
    l = np.ascontiguousarray(losses, dtype=np.float64); u = np.zeros_like(l)
    _lib.orc_snes_utilities(C.c_int(l.size), _d(l), _d(u))
    return u


def snes_update(m, s, r, losses, eta_m, eta_s):
    """Eq. 36-39: returns the updated (m, s)."""
    m = np.array(m, dtype=np.float64); s = np.array(s, dtype=np.float64)
    r = np.ascontiguousarray(r, dtype=np.float64); l = np.ascontiguousarray(losses, dtype=np.float64)
    _lib.orc_snes_update(C.c_int(r.shape[0]), C.c_int(r.shape[1]), _d(r), _d(l), C.c_double(eta_m), C.c_double(eta_s), _d(m), _d(s))
    return m, s
