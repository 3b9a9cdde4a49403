"""Thin ctypes binding over the C ABI of include/landau.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of liblandau.so.  PyTorch is used for device
memory only: device-pointer calls take torch CUDA tensors (float64 / int32, contiguous) and
return torch CUDA tensors; the *_host calls take numpy arrays and let the library do the copies.
There is NO CPU fallback: a missing library or a missing CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

from . import build as _build

_lib = None

OK = 0
NOT_CONVERGED = 1
EINVAL, ENOMEM, ECUDA, ENONFINITE, ERANGE = -1, -2, -3, -4, -5

# every symbol include/landau.h declares (tests check the .so exports exactly these)
SYMBOLS = [
    "landau_default_opts", "landau_create", "landau_destroy", "landau_eval_field",
    "landau_eval_field_host", "landau_entropy_grad", "landau_pair_field", "landau_set_markers",
    "landau_set_markers_host", "landau_get_markers", "landau_get_markers_host", "landau_step", "landau_step_dg", "landau_set_solver", "landau_set_dimension", "landau_set_step_graph", "landau_set_substep", "landau_cells_run", "landau_set_cutoff", "landau_cutoff_stats", "landau_set_mixed_precision", "landau_set_stiff_pairs", "landau_stiff_pairs_last",
    "landau_run", "landau_moments", "landau_moments_ext", "landau_get_quadrature",
    "landau_last_kernels", "landau_launch_count", "landau_profile_enable", "landau_profile_read",
    "landau_fp64_peak", "landau_fp64_peak_dmma", "landau_last_error",
    "landau_version", "landau_moments_noalloc", "landau_moments_noalloc_last_error",
    "landau_cells_max_markers",
]


class Opts(C.Structure):
    _fields_ = [("n_q", C.c_int), ("nu0", C.c_double), ("nu", C.POINTER(C.c_double)),
                ("precision", C.c_int), ("stream", C.c_void_p), ("pair_kernel", C.c_int),
                ("entropy_kernel", C.c_int), ("device", C.c_int)]


class CellInfo(C.Structure):
    _fields_ = [("status", C.c_int), ("iterations", C.c_int), ("max_iterations", C.c_int),
                ("steps_not_converged", C.c_int), ("residual", C.c_double)]


class StepInfo(C.Structure):
    _fields_ = [("iterations", C.c_int), ("residual", C.c_double), ("converged", C.c_int)]


class LandauError(RuntimeError):
    def __init__(self, code, where, msg=""):
        super().__init__(f"{where} failed with status {code}: {msg}")
        self.code = code


def library_path() -> Path:
    return _build.LIB


def load(build_if_missing: bool = True):
    """Load liblandau.so (building it with nvcc if needed).  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        _build.build()
    if not _build.LIB.exists():
        raise RuntimeError(f"{_build.LIB} is missing: build it with `python -m paper_2212_00663_b200.build` "
                           "(the CUDA path has no fallback)")
    lib = C.CDLL(str(_build.LIB))
    vp, dp, ip = C.c_void_p, C.c_void_p, C.c_void_p   # raw addresses (device or host)
    hd = C.POINTER(C.c_double)
    lib.landau_default_opts.argtypes = [C.POINTER(Opts)]
    lib.landau_default_opts.restype = None
    lib.landau_create.argtypes = [C.POINTER(vp), C.c_int, hd, hd, hd, C.POINTER(Opts)]
    lib.landau_destroy.argtypes = [vp]
    lib.landau_destroy.restype = None
    lib.landau_eval_field.argtypes = [vp, C.c_int64, dp, dp, ip, dp]
    lib.landau_eval_field_host.argtypes = [vp, C.c_int64, dp, dp, ip, dp]
    lib.landau_entropy_grad.argtypes = [vp, C.c_int64, dp, dp, ip, dp, hd]
    lib.landau_pair_field.argtypes = [vp, C.c_int64, dp, dp, ip, dp, dp]
    lib.landau_set_markers.argtypes = [vp, C.c_int64, dp, dp, ip]
    lib.landau_set_markers_host.argtypes = [vp, C.c_int64, dp, dp, ip]
    lib.landau_get_markers.argtypes = [vp, dp]
    lib.landau_get_markers_host.argtypes = [vp, dp]
    lib.landau_step.argtypes = [vp, C.c_double, C.c_double, C.c_int, C.POINTER(StepInfo)]
    lib.landau_set_solver.argtypes = [vp, C.c_int, C.c_int]
    lib.landau_set_dimension.argtypes = [vp, C.c_int]
    lib.landau_set_step_graph.argtypes = [vp, C.c_int]
    lib.landau_set_substep.argtypes = [vp, C.c_int]
    lib.landau_set_cutoff.argtypes = [vp, C.c_int, C.c_int]
    lib.landau_set_mixed_precision.argtypes = [vp, C.c_double]
    lib.landau_set_stiff_pairs.argtypes = [vp, C.c_double]
    lib.landau_stiff_pairs_last.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    lib.landau_cutoff_stats.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    lib.landau_cells_run.argtypes = [vp, C.c_int, vp, vp, vp, vp, vp, C.c_int, C.c_double, C.c_double, C.c_int,
                                     C.POINTER(CellInfo)]
    lib.landau_step_dg.argtypes = [vp, C.c_double, C.c_double, C.c_int, C.POINTER(StepInfo)]
    lib.landau_run.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_int, C.POINTER(StepInfo)]
    lib.landau_moments.argtypes = [vp, hd, hd, hd, hd]
    lib.landau_moments_ext.argtypes = [vp, hd, hd]
    lib.landau_get_quadrature.argtypes = [vp, hd, hd]
    lib.landau_last_kernels.argtypes = [vp]
    lib.landau_last_kernels.restype = C.c_char_p
    lib.landau_launch_count.argtypes = [vp]
    lib.landau_launch_count.restype = C.c_int64
    lib.landau_profile_enable.argtypes = [vp, C.c_int]
    lib.landau_profile_read.argtypes = [vp, hd, C.POINTER(C.c_int64), hd, C.POINTER(C.c_int64)]
    lib.landau_fp64_peak.argtypes = [vp, C.c_int, hd]
    lib.landau_fp64_peak_dmma.argtypes = [vp, C.c_int, hd]
    lib.landau_last_error.argtypes = [vp]
    lib.landau_last_error.restype = C.c_char_p
    lib.landau_version.restype = C.c_char_p
    lib.landau_cells_max_markers.argtypes = [C.c_int]
    lib.landau_moments_noalloc.argtypes = [C.c_int64, dp, dp, ip, C.c_int, hd, dp, vp]
    lib.landau_moments_noalloc_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def _hd(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


MOMENTS_NOALLOC_MAX_N = 1 << 21


def cells_max_markers(n_q: int) -> int:
    """Largest cell landau_cells_run accepts at this n_q (host-side query, no GPU needed)."""
    return int(load().landau_cells_max_markers(int(n_q)))


def moments_noalloc(v, w, sid, mass, out, stream=None, N=None):
    """n_s, P_s, K_s per species without a context and without any device allocation by the library
    (landau_moments_noalloc, include/landau.h): for callers that cannot cudaMalloc -- HBM already fully
    owned by the host code, or a hook inside an asynchronous loop that must not synchronise the device.

    v [N, 3] float64, w [N] float64, sid [N] int32 and out [S, 5] float64 are CUDA tensors the CALLER
    made (this wrapper creates none, so that the whole call allocates nothing); mass is a host
    sequence of S masses.  Asynchronous on `stream` (default: torch's current stream); `out` holds
    n, Px, Py, Pz, K per row once the stream has passed the call.  At most MOMENTS_NOALLOC_MAX_N
    markers and 16 species: beyond that the library refuses (LandauError, code EINVAL).  All calls on
    a device share one built-in scratch array: do not let two of them overlap on the GPU.  Call it
    once at start-up, outside stream capture (the first call per device does the set-up)."""
    import torch

    lib = load()
    m = _f64(mass)
    for t_, dt_ in ((v, torch.float64), (w, torch.float64), (sid, torch.int32), (out, torch.float64)):
        if not (t_.is_cuda and t_.dtype == dt_ and t_.is_contiguous()):
            raise ValueError("moments_noalloc takes contiguous CUDA tensors (float64 / int32) made by the caller")
    n = int(w.shape[0]) if N is None else int(N)
    if out.numel() < 5 * m.shape[0]:
        raise ValueError("out must hold n_species x 5 doubles")
    st = torch.cuda.current_stream(w.device).cuda_stream if stream is None else int(
        stream.cuda_stream if hasattr(stream, "cuda_stream") else stream)
    with torch.cuda.device(w.device):
        rc = lib.landau_moments_noalloc(n, v.data_ptr(), w.data_ptr(), sid.data_ptr(), int(m.shape[0]), _hd(m),
                                        out.data_ptr(), C.c_void_p(st))
    if rc:
        raise LandauError(rc, "landau_moments_noalloc", lib.landau_moments_noalloc_last_error().decode())
    return out


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Landau:
    """One context = one species table + one CUDA stream (+ optionally held markers)."""

    def __init__(self, mass, charge, eps, n_q: int = 4, nu0: float = 1.0, nu=None, precision: int = 0,
                 stream=None, pair_kernel: int = 0, entropy_kernel: int = 0, device: int = -1):
        import torch  # device memory + streams only

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2212_00663_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self._lib = load()
        self.mass, self.charge, self.eps = _f64(mass), _f64(charge), _f64(eps)
        self.S = int(self.mass.shape[0])
        self.n_q = int(n_q)
        o = Opts()
        self._lib.landau_default_opts(C.byref(o))
        o.n_q, o.nu0, o.precision = int(n_q), float(nu0), int(precision)
        o.pair_kernel, o.entropy_kernel, o.device = int(pair_kernel), int(entropy_kernel), int(device)
        self._nu = None if nu is None else _f64(nu)
        if self._nu is not None:
            o.nu = _hd(self._nu)
        if stream is not None:
            o.stream = C.c_void_p(int(stream.cuda_stream if hasattr(stream, "cuda_stream") else stream))
        self._dev = torch.device("cuda", torch.cuda.current_device() if device < 0 else device)
        h = C.c_void_p()
        rc = self._lib.landau_create(C.byref(h), self.S, _hd(self.mass), _hd(self.charge), _hd(self.eps), C.byref(o))
        if rc:
            raise LandauError(rc, "landau_create")
        self._h = h
        self.N = 0

    # -- plumbing ---------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            self._lib.landau_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, where, allow=(0,)):
        if rc not in allow:
            raise LandauError(rc, where, self._lib.landau_last_error(self._h).decode())
        return rc

    def _dev_in(self, v, w, sid):
        t = self._torch
        v = t.as_tensor(v, dtype=t.float64, device=self._dev).contiguous()
        w = t.as_tensor(w, dtype=t.float64, device=self._dev).contiguous()
        sid = t.as_tensor(sid, dtype=t.int32, device=self._dev).contiguous()
        return v, w, sid, int(w.shape[0])

    def last_kernels(self) -> str:
        return self._lib.landau_last_kernels(self._h).decode()

    def launch_count(self) -> int:
        return int(self._lib.landau_launch_count(self._h))

    def quadrature(self):
        k, a = np.empty(self.n_q), np.empty(self.n_q)
        self._check(self._lib.landau_get_quadrature(self._h, _hd(k), _hd(a)), "landau_get_quadrature")
        return k, a

    # -- field ------------------------------------------------------------------------------
    def eval_field(self, v, w, sid):
        v, w, sid, N = self._dev_in(v, w, sid)
        out = self._torch.empty((N, 3), dtype=self._torch.float64, device=self._dev)
        self._check(self._lib.landau_eval_field(self._h, N, v.data_ptr(), w.data_ptr(), sid.data_ptr(),
                                                out.data_ptr()), "landau_eval_field")
        return out

    def eval_field_host(self, v, w, sid):
        v, w = _f64(v), _f64(w)
        sid = np.ascontiguousarray(sid, dtype=np.int32)
        out = np.empty((w.shape[0], 3))
        self._check(self._lib.landau_eval_field_host(self._h, w.shape[0], v.ctypes.data, w.ctypes.data,
                                                     sid.ctypes.data, out.ctypes.data), "landau_eval_field_host")
        return out

    def entropy_grad(self, v, w, sid, with_entropy: bool = False):
        v, w, sid, N = self._dev_in(v, w, sid)
        G = self._torch.empty((N, 3), dtype=self._torch.float64, device=self._dev)
        S = np.empty(self.S)
        self._check(self._lib.landau_entropy_grad(self._h, N, v.data_ptr(), w.data_ptr(), sid.data_ptr(),
                                                  G.data_ptr(), _hd(S) if with_entropy else None),
                    "landau_entropy_grad")
        return (G, S) if with_entropy else G

    def pair_field(self, v, w, sid, G):
        v, w, sid, N = self._dev_in(v, w, sid)
        G = self._torch.as_tensor(G, dtype=self._torch.float64, device=self._dev).contiguous()
        out = self._torch.empty((N, 3), dtype=self._torch.float64, device=self._dev)
        self._check(self._lib.landau_pair_field(self._h, N, v.data_ptr(), w.data_ptr(), sid.data_ptr(),
                                                G.data_ptr(), out.data_ptr()), "landau_pair_field")
        return out

    # -- stepping ---------------------------------------------------------------------------
    def set_markers(self, v, w, sid):
        v, w, sid, N = self._dev_in(v, w, sid)
        self._check(self._lib.landau_set_markers(self._h, N, v.data_ptr(), w.data_ptr(), sid.data_ptr()),
                    "landau_set_markers")
        self.N = N

    def set_markers_host(self, v, w, sid):
        v, w = _f64(v), _f64(w)
        sid = np.ascontiguousarray(sid, dtype=np.int32)
        self._check(self._lib.landau_set_markers_host(self._h, w.shape[0], v.ctypes.data, w.ctypes.data,
                                                      sid.ctypes.data), "landau_set_markers_host")
        self.N = int(w.shape[0])

    def get_markers(self):
        out = self._torch.empty((self.N, 3), dtype=self._torch.float64, device=self._dev)
        self._check(self._lib.landau_get_markers(self._h, out.data_ptr()), "landau_get_markers")
        return out

    def get_markers_host(self):
        out = np.empty((self.N, 3))
        self._check(self._lib.landau_get_markers_host(self._h, out.ctypes.data), "landau_get_markers_host")
        return out

    def step(self, dt, tol=1e-12, max_iter=50):
        """Returns (status, iterations, residual, converged); status 1 = not converged."""
        info = StepInfo()
        rc = self._check(self._lib.landau_step(self._h, float(dt), float(tol), int(max_iter), C.byref(info)),
                         "landau_step", allow=(0, 1))
        return rc, int(info.iterations), float(info.residual), bool(info.converged)

    def set_solver(self, solver: int = 0, depth: int = 3):
        """0 = the paper's Jacobi fixed point (default); 1 = Anderson acceleration of depth 1..10; 2 = Jacobian-free
        Newton-Krylov with GMRES restart length `depth` 1..30 (NEXT-4)."""
        self._check(self._lib.landau_set_solver(self._h, int(solver), int(depth)), "landau_set_solver")

    def cells_run(self, cell_offset, v, w, sid, n_steps, dt, tol=1e-12, max_iter=50, out=None, strict=True):
        """Many collision cells in one launch (NEXT-3).  cell_offset: host int64 [n_cells + 1]; v, w, sid: the
        markers of all cells (device tensors or arrays).  Returns (status, v_out tensor, info record array with
        fields status / iterations / max_iterations / steps_not_converged / residual).  strict=False returns a
        negative status (some cell was rejected and copied through) instead of raising; see info["status"]."""
        off = np.ascontiguousarray(cell_offset, dtype=np.int64)
        n_cells = int(off.shape[0] - 1)
        v, w, sid, N = self._dev_in(v, w, sid)
        if out is None:
            out = self._torch.empty((N, 3), dtype=self._torch.float64, device=self._dev)
        infos = (CellInfo * n_cells)()
        rc = self._check(self._lib.landau_cells_run(self._h, n_cells, off.ctypes.data, v.data_ptr(), w.data_ptr(),
                                                    sid.data_ptr(), out.data_ptr(), int(n_steps), float(dt),
                                                    float(tol), int(max_iter), infos),
                         "landau_cells_run", allow=(0, 1) if strict else (0, 1, EINVAL, ENONFINITE, ERANGE))
        info = np.array([(i.status, i.iterations, i.max_iterations, i.steps_not_converged, i.residual) for i in infos],
                        dtype=[("status", "i4"), ("iterations", "i4"), ("max_iterations", "i4"),
                               ("steps_not_converged", "i4"), ("residual", "f8")])
        return rc, out, info

    def set_step_graph(self, mode: int = 1):
        """0 = plain launch sequence; 1 (default) = launch-bound clouds run all iterations of a step in one persistent
        kernel, other small clouds replay the step as a CUDA graph; 2 = CUDA-graph step always."""
        self._check(self._lib.landau_set_step_graph(self._h, int(mode)), "landau_set_step_graph")

    def set_substep(self, max_halvings: int = 0):
        """0 = commit unconverged steps (the paper's behaviour); k > 0 = redo them as two half steps, up to k levels."""
        self._check(self._lib.landau_set_substep(self._h, int(max_halvings)), "landau_set_substep")

    def set_stiff_pairs(self, theta: float = 0.0):
        """> 0: pairs with stiffness L_pq > theta are solved implicitly and exactly inside the fixed-point iteration
        (same Eq. (24); NEXT-4 robustness); 0 = off (the paper's plain iteration)."""
        self._check(self._lib.landau_set_stiff_pairs(self._h, float(theta)), "landau_set_stiff_pairs")

    def stiff_pairs_last(self):
        """(pairs treated by the last step, overflow flag)."""
        a, b = C.c_int(0), C.c_int(0)
        self._check(self._lib.landau_stiff_pairs_last(self._h, C.byref(a), C.byref(b)), "landau_stiff_pairs_last")
        return int(a.value), int(b.value)

    def set_mixed_precision(self, f32_until: float = 0.0):
        """> 0: pass 2 of the implicit step runs in FP32 while the residual exceeds f32_until (then FP64); 0 = off."""
        self._check(self._lib.landau_set_mixed_precision(self._h, float(f32_until)), "landau_set_mixed_precision")

    def set_cutoff(self, on: bool = True, morton: bool = True):
        """Gaussian cutoff of pass 1 (NEXT-4): skip source tiles that cannot change a node sum by 2^-60 relative;
        morton: bucket every species along a Morton curve at pack time so that tiles are compact."""
        self._check(self._lib.landau_set_cutoff(self._h, int(bool(on)), int(bool(morton))), "landau_set_cutoff")

    def cutoff_stats(self):
        """(source tiles considered, skipped) by the last pass 1."""
        a, b = C.c_int64(0), C.c_int64(0)
        self._check(self._lib.landau_cutoff_stats(self._h, C.byref(a), C.byref(b)), "landau_cutoff_stats")
        return int(a.value), int(b.value)

    def set_dimension(self, dim: int = 3):
        """3 (default) or 2 = the paper's 2-V setting: v_z = 0 is preserved exactly (NEXT-2)."""
        self._check(self._lib.landau_set_dimension(self._h, int(dim)), "landau_set_dimension")

    def step_dg(self, dt, tol=1e-12, max_iter=50):
        """Discrete-gradient step, Eqs. (46)-(49).  Returns as step()."""
        info = StepInfo()
        rc = self._check(self._lib.landau_step_dg(self._h, float(dt), float(tol), int(max_iter), C.byref(info)),
                         "landau_step_dg", allow=(0, 1))
        return rc, int(info.iterations), float(info.residual), bool(info.converged)

    def run(self, n_steps, dt, tol=1e-12, max_iter=50):
        """n_steps steps, one host sync.  Returns (status, [(iterations, residual, converged)])."""
        infos = (StepInfo * int(n_steps))()
        rc = self._check(self._lib.landau_run(self._h, int(n_steps), float(dt), float(tol), int(max_iter), infos),
                         "landau_run", allow=(0, 1))
        return rc, [(int(i.iterations), float(i.residual), bool(i.converged)) for i in infos]

    def moments(self, with_entropy: bool = True):
        n, P, K, S = np.empty(self.S), np.empty((self.S, 3)), np.empty(self.S), np.empty(self.S)
        self._check(self._lib.landau_moments(self._h, _hd(n), _hd(P), _hd(K), _hd(S) if with_entropy else None),
                    "landau_moments")
        return dict(n=n, P=P, K=K, S_eps=S if with_entropy else None)

    def moments_ext(self):
        stress, m4 = np.empty((self.S, 6)), np.empty((self.S, 3))
        self._check(self._lib.landau_moments_ext(self._h, _hd(stress), _hd(m4)), "landau_moments_ext")
        return stress, m4

    def profile_enable(self, on: bool = True):
        self._check(self._lib.landau_profile_enable(self._h, int(bool(on))), "landau_profile_enable")

    def profile_read(self):
        """dict(pair_ms, pair_launches, entropy_ms, entropy_launches) since profile_enable."""
        pm, em = C.c_double(0.0), C.c_double(0.0)
        pn, en = C.c_int64(0), C.c_int64(0)
        self._check(self._lib.landau_profile_read(self._h, C.byref(pm), C.byref(pn), C.byref(em), C.byref(en)),
                    "landau_profile_read")
        return dict(pair_ms=pm.value, pair_launches=pn.value, entropy_ms=em.value, entropy_launches=en.value)

    def fp64_peak_dmma(self, reps: int = 5) -> float:
        out = C.c_double(0.0)
        self._check(self._lib.landau_fp64_peak_dmma(self._h, int(reps), C.byref(out)), "landau_fp64_peak_dmma")
        return float(out.value)

    def fp64_peak(self, reps: int = 5) -> float:
        out = C.c_double(0.0)
        self._check(self._lib.landau_fp64_peak(self._h, int(reps), C.byref(out)), "landau_fp64_peak")
        return float(out.value)
