"""Thin Python binding of libnep_b200.so (include/nep_b200.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/nep_b200.cu; PyTorch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing, loading fails."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libnep_b200.so")
_lib = None

SYMBOLS = ["nep_create", "nep_create_ex", "nep_descriptor_dim", "nep_num_params", "nep_destroy", "nep_workspace_bytes",
           "nep_system_create", "nep_system_destroy", "nep_system_set_path", "nep_system_path", "nep_neighbors", "nep_get_neighbors", "nep_compute", "nep_compute_internals",
           "nep_md_step", "nep_md_step_driven", "nep_status", "nep_stats", "nep_launch_count", "nep_profile", "nep_get_profile", "nep_measure_fp32_peak", "nep_measure_fp32_patterns",
           "nep_trainer_workspace_bytes", "nep_trainer_create", "nep_trainer_destroy", "nep_trainer_num_params", "nep_trainer_status",
           "nep_trainer_losses", "nep_trainer_predict", "nep_snes_sample", "nep_snes_update", "nep_loss_noalloc",
           "nep_strerror"]


class NepError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__("%s failed: %d (%s)" % (where, code, lib().nep_strerror(code).decode()))


class Hyper(C.Structure):
    _fields_ = [("rc_radial", C.c_double), ("rc_angular", C.c_double), ("n_max_radial", C.c_int),
                ("n_max_angular", C.c_int), ("l_max", C.c_int), ("n_neurons", C.c_int), ("n_types", C.c_int)]


class HyperEx(C.Structure):
    _fields_ = [("base", Hyper), ("n_hidden_layers", C.c_int), ("n_neurons_2", C.c_int), ("n_neurons_3", C.c_int),
                ("angular_kind", C.c_int)]


def lib():
    """Loads the C-ABI library (built by paper_2107_08119_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError("libnep_b200.so is missing: run `python -m paper_2107_08119_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        L.nep_strerror.restype = C.c_char_p
        L.nep_workspace_bytes.restype = C.c_size_t
        L.nep_workspace_bytes.argtypes = [C.c_void_p, C.c_int64, C.c_int, C.c_int, C.c_double]
        L.nep_create.argtypes = [C.POINTER(Hyper), C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(C.c_void_p)]
        L.nep_create_ex.argtypes = [C.POINTER(HyperEx), C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(C.c_void_p)]
        L.nep_system_create.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_void_p,
                                        C.c_size_t, C.POINTER(C.c_void_p)]
        L.nep_neighbors.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nep_get_neighbors.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nep_compute.argtypes = [C.c_void_p] * 8
        L.nep_compute_internals.argtypes = [C.c_void_p] * 6
        L.nep_md_step.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_int] + [C.c_void_p] * 7
        L.nep_md_step_driven.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_int] + [C.c_void_p] * 10
        for f in ("nep_destroy", "nep_system_destroy"):
            getattr(L, f).argtypes = [C.c_void_p]
            getattr(L, f).restype = None
        for f in ("nep_descriptor_dim", "nep_num_params", "nep_status"):
            getattr(L, f).argtypes = [C.c_void_p]
        L.nep_stats.argtypes = [C.c_void_p, C.c_void_p]
        L.nep_system_set_path.argtypes = [C.c_void_p, C.c_int]
        L.nep_system_path.argtypes = [C.c_void_p]
        L.nep_launch_count.argtypes = [C.c_void_p]
        L.nep_launch_count.restype = C.c_int64
        L.nep_profile.argtypes = [C.c_void_p, C.c_int]
        L.nep_trainer_workspace_bytes.restype = C.c_size_t
        L.nep_trainer_workspace_bytes.argtypes = [C.POINTER(HyperEx), C.c_int, C.c_int64, C.c_int, C.c_int]
        L.nep_trainer_create.argtypes = [C.POINTER(HyperEx), C.c_void_p, C.c_int] + [C.c_void_p] * 7 + [C.c_int, C.c_int, C.c_void_p,
                                          C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]
        L.nep_trainer_destroy.argtypes = [C.c_void_p]; L.nep_trainer_destroy.restype = None
        L.nep_trainer_num_params.argtypes = [C.c_void_p]; L.nep_trainer_status.argtypes = [C.c_void_p]
        L.nep_trainer_losses.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nep_trainer_predict.argtypes = [C.c_void_p] * 6
        L.nep_snes_sample.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.nep_snes_update.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double,
                                      C.c_double, C.c_void_p]
        L.nep_get_profile.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.nep_loss_noalloc.argtypes = [C.c_int64, C.c_int64, C.c_int64] + [C.c_void_p] * 10 + [C.c_char_p, C.c_size_t]
        _lib = L
    return _lib


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _check(code, where):
    if code != 0:
        raise NepError(code, where)


class Model:
    """nep_create / nep_destroy."""

    def __init__(self, rc_radial, rc_angular, n_max_radial, n_max_angular, l_max, n_neurons, atomic_numbers, params,
                 hidden_layers=None, angular_kind=0):
        """hidden_layers: None (one layer of n_neurons) or a list of 1..3 widths; angular_kind 1: q_nn'l (nep_create_ex)."""
        zs = np.ascontiguousarray(atomic_numbers, dtype=np.int32)
        par = np.ascontiguousarray(params, dtype=np.float64)
        self.hyper = Hyper(rc_radial, rc_angular, n_max_radial, n_max_angular, l_max, n_neurons, len(zs))
        self._h = C.c_void_p()
        if hidden_layers is None and angular_kind == 0:
            _check(lib().nep_create(C.byref(self.hyper), zs.ctypes.data_as(C.c_void_p), par.ctypes.data_as(C.c_void_p),
                                    par.size, C.byref(self._h)), "nep_create")
        else:
            w = list(hidden_layers) if hidden_layers is not None else [n_neurons]
            self.hyper.n_neurons = w[0]
            hx = HyperEx(self.hyper, len(w), w[1] if len(w) > 1 else 0, w[2] if len(w) > 2 else 0, angular_kind)
            _check(lib().nep_create_ex(C.byref(hx), zs.ctypes.data_as(C.c_void_p), par.ctypes.data_as(C.c_void_p),
                                       par.size, C.byref(self._h)), "nep_create_ex")

    @property
    def descriptor_dim(self):
        return lib().nep_descriptor_dim(self._h)

    @property
    def num_params(self):
        return lib().nep_num_params(self._h)

    def __del__(self):
        if getattr(self, "_h", None) and self._h.value and _lib is not None:
            _lib.nep_destroy(self._h)
            self._h = C.c_void_p()


class System:
    """nep_system_create + the compute calls.  Tensors are CUDA tensors owned by the caller."""

    def __init__(self, model: Model, types: torch.Tensor, cap_radial=64, cap_angular=32, skin=1.0):
        assert types.is_cuda and types.dtype == torch.int32
        self.model = model
        self.n = types.numel()
        self.cap_radial, self.cap_angular, self.skin = cap_radial, cap_angular, skin
        nbytes = lib().nep_workspace_bytes(model._h, self.n, cap_radial, cap_angular, skin)
        if nbytes == 0:
            raise NepError(-1, "nep_workspace_bytes")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=types.device)
        off = (-self.workspace.data_ptr()) % 256
        self._h = C.c_void_p()
        _check(lib().nep_system_create(model._h, self.n, _ptr(types), cap_radial, cap_angular, float(skin),
                                       C.c_void_p(self.workspace.data_ptr() + off), nbytes, C.byref(self._h)),
               "nep_system_create")

    PATH_AUTO, PATH_THREAD, PATH_GROUP = 0, 1, 2

    def set_path(self, path: int):
        """nep_system_set_path: 0 auto, 1 one thread per atom (k_main), 2 16 lanes per atom (k_gen)."""
        _check(lib().nep_system_set_path(self._h, int(path)), "nep_system_set_path")

    @property
    def path(self):
        return lib().nep_system_path(self._h)

    def neighbors(self, pos: torch.Tensor, box):
        assert pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous() and pos.shape == (3, self.n)
        b = (C.c_double * 3)(*[float(v) for v in box])
        _check(lib().nep_neighbors(self._h, _ptr(pos), C.cast(b, C.c_void_p), _stream()), "nep_neighbors")

    def get_neighbors(self, which: int):
        cap = self.cap_angular if which else self.cap_radial
        count = torch.empty(self.n, dtype=torch.int32, device=self.workspace.device)
        index = torch.empty((self.n, cap), dtype=torch.int32, device=self.workspace.device)
        _check(lib().nep_get_neighbors(self._h, which, _ptr(count), _ptr(index), _stream()), "nep_get_neighbors")
        return count, index

    def alloc_outputs(self):
        dev = self.workspace.device
        return (torch.empty(self.n, dtype=torch.float32, device=dev), torch.empty((3, self.n), dtype=torch.float32, device=dev),
                torch.empty((9, self.n), dtype=torch.float32, device=dev), torch.empty((3, self.n), dtype=torch.float32, device=dev))

    def compute(self, pos, vel=None, out=None):
        assert pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous()
        U, F, W, J = out if out is not None else self.alloc_outputs()
        _check(lib().nep_compute(self._h, _ptr(pos), _ptr(vel), _ptr(U), _ptr(F), _ptr(W), _ptr(J), _stream()),
               "nep_compute")
        return U, F, W, J

    def compute_internals(self, pos):
        """(q [D,N], dU/dq [D,N], p [N,cap_radial,3]) of the intermediate rows, for parity tests."""
        dev = self.workspace.device
        D = self.model.descriptor_dim
        q = torch.zeros((D, self.n), dtype=torch.float32, device=dev)
        fp = torch.zeros((D, self.n), dtype=torch.float32, device=dev)
        p = torch.zeros((self.n, self.cap_radial, 3), dtype=torch.float32, device=dev)
        _check(lib().nep_compute_internals(self._h, _ptr(pos), _ptr(q), _ptr(fp), _ptr(p), _stream()), "nep_compute_internals")
        return q, fp, p

    def md_step(self, pos, vel, masses, dt, n_steps, out=None, heat_sum=None, thermo=None):
        assert pos.dtype == torch.float64 and vel.dtype == torch.float64 and pos.is_contiguous() and vel.is_contiguous()
        U, F, W, J = out if out is not None else self.alloc_outputs()
        m = np.ascontiguousarray(masses, dtype=np.float64)
        _check(lib().nep_md_step(self._h, _ptr(pos), _ptr(vel), m.ctypes.data_as(C.c_void_p), float(dt), int(n_steps),
                                 _ptr(U), _ptr(F), _ptr(W), _ptr(J), _ptr(heat_sum), _ptr(thermo), _stream()),
               "nep_md_step")
        return U, F, W, J

    def md_step_driven(self, pos, vel, masses, dt, n_steps, driving_force, out=None, heat_sum=None, thermo=None, w0=None, kt=None):
        """nep_md_step_driven: HNEMD driving force F_e (Eq. 9) and K(t) = sum_i W_i(0) . v_i(t) (Eq. 11)."""
        assert pos.dtype == torch.float64 and vel.dtype == torch.float64 and pos.is_contiguous() and vel.is_contiguous()
        U, F, W, J = out if out is not None else self.alloc_outputs()
        m = np.ascontiguousarray(masses, dtype=np.float64)
        fe = None if driving_force is None else np.ascontiguousarray(driving_force, dtype=np.float64)
        _check(lib().nep_md_step_driven(self._h, _ptr(pos), _ptr(vel), m.ctypes.data_as(C.c_void_p), float(dt), int(n_steps),
                                        None if fe is None else fe.ctypes.data_as(C.c_void_p),
                                        _ptr(U), _ptr(F), _ptr(W), _ptr(J), _ptr(heat_sum), _ptr(thermo), _ptr(w0), _ptr(kt),
                                        _stream()), "nep_md_step_driven")
        return U, F, W, J

    def status(self):
        """Synchronises; raises NepError on a sticky device-side error (overflow, stale list)."""
        _check(lib().nep_status(self._h), "nep_status")

    def stats(self):
        out = (C.c_int64 * 4)()
        _check(lib().nep_stats(self._h, C.cast(out, C.c_void_p)), "nep_stats")
        return dict(rebuilds=out[0], max_radial=out[1], max_angular=out[2], max_verlet=out[3])

    PHASES = ("kick_drift", "build", "filter", "main", "assemble", "state")

    def launch_count(self):
        return lib().nep_launch_count(self._h)

    def profile(self, enable: bool):
        _check(lib().nep_profile(self._h, int(enable)), "nep_profile")

    def get_profile(self):
        ms = (C.c_double * 8)(); cnt = (C.c_int64 * 8)()
        _check(lib().nep_get_profile(self._h, C.cast(ms, C.c_void_p), C.cast(cnt, C.c_void_p)), "nep_get_profile")
        return {name: dict(ms=ms[k], count=cnt[k]) for k, name in enumerate(self.PHASES)}

    def __del__(self):
        if getattr(self, "_h", None) and self._h.value and _lib is not None:
            _lib.nep_system_destroy(self._h)
            self._h = C.c_void_p()


def measure_fp32_peak():
    """(TFLOP/s with scalar FFMA, TFLOP/s with packed fma.f32x2) from the library's FMA-chain microbenchmark."""
    a, b = C.c_double(), C.c_double()
    _check(lib().nep_measure_fp32_peak(C.byref(a), C.byref(b), _stream()), "nep_measure_fp32_peak")
    return a.value, b.value


def measure_fp32_patterns():
    """TFLOP/s of (FFMA with three distinct registers, packed descriptor contraction, packed force contraction)."""
    out = (C.c_double * 3)()
    _check(lib().nep_measure_fp32_patterns(C.cast(out, C.c_void_p), _stream()), "nep_measure_fp32_patterns")
    return out[0], out[1], out[2]


def from_workload(w, cap_radial=64, cap_angular=32, skin=1.0, device="cuda:0", path=None):
    """Model + System + device tensors for a paper_2107_08119_b200.inputs.Workload (path: nep_system_set_path)."""
    model = Model(w.rc_r, w.rc_a, w.n_max_r, w.n_max_a, w.l_max, w.n_neurons, w.atomic_numbers, w.params)
    types = torch.from_numpy(w.types).to(device)
    system = System(model, types, cap_radial, cap_angular, skin)
    if path is not None:
        system.set_path(path)
    pos = torch.from_numpy(w.pos).to(device).contiguous()
    vel = torch.from_numpy(w.vel).to(device).contiguous()
    return model, system, pos, vel


class Trainer:
    """nep_trainer_*: the loss of Eq. 29-34 for a population over concatenated structures, and SNES (Eq. 35-39)."""

    def __init__(self, rc_radial, rc_angular, n_max_radial, n_max_angular, l_max, hidden_layers, first, boxes, pos,
                 e_tar=None, f_tar=None, v_tar=None, angular_kind=0, cap_radial=64, cap_angular=32, types=None,
                 atomic_numbers=(14,)):
        w = list(hidden_layers)
        zs = np.ascontiguousarray(atomic_numbers, dtype=np.int32)
        base = Hyper(rc_radial, rc_angular, n_max_radial, n_max_angular, l_max, w[0], len(zs))
        self.hx = HyperEx(base, len(w), w[1] if len(w) > 1 else 0, w[2] if len(w) > 2 else 0, angular_kind)
        first = np.ascontiguousarray(first, dtype=np.int64); boxes = np.ascontiguousarray(boxes, dtype=np.float64)
        self.n_structures, self.n = len(first) - 1, int(first[-1])
        assert pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous() and pos.shape == (3, self.n)
        self._keep = (pos, e_tar, f_tar, v_tar, types)       # the library keeps the target pointers
        nbytes = lib().nep_trainer_workspace_bytes(C.byref(self.hx), self.n_structures, self.n, cap_radial, cap_angular)
        if nbytes == 0:
            raise NepError(-1, "nep_trainer_workspace_bytes")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=pos.device)
        off = (-self.workspace.data_ptr()) % 256
        self._h = C.c_void_p()
        _check(lib().nep_trainer_create(C.byref(self.hx), zs.ctypes.data_as(C.c_void_p), self.n_structures,
                                        first.ctypes.data_as(C.c_void_p), boxes.ctypes.data_as(C.c_void_p), _ptr(pos), _ptr(types),
                                        _ptr(e_tar), _ptr(f_tar), _ptr(v_tar),
                                        cap_radial, cap_angular, C.c_void_p(self.workspace.data_ptr() + off), nbytes, _stream(),
                                        C.byref(self._h)), "nep_trainer_create")
        self.num_params = lib().nep_trainer_num_params(self._h)

    def losses(self, z, lambdas):
        """z [n_pop, N_par] fp64 cuda -> [n_pop, 6] = L_e, L_f, L_v, L_1, L_2, L."""
        assert z.is_cuda and z.dtype == torch.float64 and z.is_contiguous() and z.shape[1] == self.num_params
        lam = np.ascontiguousarray(lambdas, dtype=np.float64)
        out = torch.zeros((z.shape[0], 6), dtype=torch.float64, device=z.device)
        _check(lib().nep_trainer_losses(self._h, _ptr(z), z.shape[0], lam.ctypes.data_as(C.c_void_p), _ptr(out), _stream()),
               "nep_trainer_losses")
        return out

    def predict(self, z):
        dev = z.device
        e = torch.zeros(self.n_structures, dtype=torch.float32, device=dev)
        f = torch.zeros((3, self.n), dtype=torch.float32, device=dev)
        v = torch.zeros((self.n_structures, 6), dtype=torch.float32, device=dev)
        _check(lib().nep_trainer_predict(self._h, _ptr(z), _ptr(e), _ptr(f), _ptr(v), _stream()), "nep_trainer_predict")
        return e, f, v

    def status(self):
        _check(lib().nep_trainer_status(self._h), "nep_trainer_status")

    def __del__(self):
        if getattr(self, "_h", None) and self._h.value and _lib is not None:
            _lib.nep_trainer_destroy(self._h)
            self._h = C.c_void_p()


def snes_sample(m, s, r):
    z = torch.empty_like(r)
    _check(lib().nep_snes_sample(_ptr(m), _ptr(s), _ptr(r), r.shape[0], r.shape[1], _ptr(z), _stream()), "nep_snes_sample")
    return z


def snes_update(m, s, r, loss, eta_m, eta_s):
    """In place on m, s; loss: [n_pop] or [n_pop, 6] (the total is column 5)."""
    stride = 1 if loss.dim() == 1 else loss.shape[1]
    ptr = loss.data_ptr() + (0 if loss.dim() == 1 else 5 * loss.element_size())
    _check(lib().nep_snes_update(_ptr(m), _ptr(s), _ptr(r), C.c_void_p(ptr), stride, r.shape[0], r.shape[1], float(eta_m),
                                 float(eta_s), _stream()), "nep_snes_update")


def loss_noalloc(e, f, v, e_tar, f_tar, v_tar, z, lambdas, out):
    """nep_loss_noalloc: Eq. 29-34 for one parameter vector from predictions on the device, for callers that cannot
    allocate device memory (see include/nep_b200.h for who they are and for the limits: a fixed 0.5 MiB scratch inside
    the library, 3 N + 7 S + n_par <= 16,777,216, first call per device before any stream capture, no overlapping
    calls).  Nothing is allocated here either: `out` [6] fp64 cuda is the caller's.  e [S], f [3, N], v [S, 6] and the
    targets: fp32 cuda, contiguous; z [n_par] fp64 cuda.  Returns out = L_e, L_f, L_v, L_1, L_2, L."""
    for t in (e, f, v, e_tar, f_tar, v_tar):
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
    assert z.is_cuda and z.dtype == torch.float64 and z.is_contiguous() and z.dim() == 1
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 6
    S, N = e.shape[0], f.shape[1]
    assert f.shape == (3, N) and v.shape == (S, 6) and e_tar.shape == e.shape and f_tar.shape == f.shape and v_tar.shape == v.shape
    lam = np.ascontiguousarray(lambdas, dtype=np.float64)
    msg = C.create_string_buffer(512)
    code = lib().nep_loss_noalloc(S, N, z.shape[0], _ptr(e), _ptr(f), _ptr(v), _ptr(e_tar), _ptr(f_tar), _ptr(v_tar), _ptr(z),
                                  lam.ctypes.data_as(C.c_void_p), _ptr(out), _stream(), msg, len(msg))
    if code != 0:
        raise NepError(code, msg.value.decode() or "nep_loss_noalloc")
    return out
