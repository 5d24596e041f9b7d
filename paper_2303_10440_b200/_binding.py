"""ctypes binding of include/deltamic.h.  Same names as the C ABI, argument marshalling only."""
from __future__ import annotations

import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(HERE, "libdeltamic.so")

DM_VOLUME, DM_SURFACE = 0, 1
DM_OPT_FORWARD_PATH, DM_OPT_BACKWARD_PATH, DM_OPT_TAU, DM_OPT_TAU_BWD, DM_OPT_AREA_NORMALISED = 0, 1, 2, 3, 4
DM_OPT_REUSE_SPECTRUM = 5

# every symbol include/deltamic.h declares
_SYMBOLS = (
    "dm_plan_create", "dm_plan_set_stream", "dm_plan_set_slab", "dm_plan_set_narrow_band", "dm_plan_set_face_weights", "dm_plan_update_face_weights", "dm_plan_set_option", "dm_mesh_ft_forward", "dm_mesh_ft_backward", "dm_mesh_ft_backward_with_spectrum", "dm_render",
    "dm_render_backward", "dm_spectrum_to_image", "dm_image_to_spectrum_cotangent", "dm_plan_stage_ms",
    "dm_plan_launch_count", "dm_plan_paths_used", "dm_plan_destroy", "dm_error_string", "dm_version",
    "dm_shape_params_default", "dm_shape_state_create", "dm_shape_precondition", "dm_shape_last_cg_iterations", "dm_shape_last_cg_residuals", "dm_shape_step", "dm_shape_state_destroy",
    "dm_mesh_ft_forward_noalloc",
)
DM_NOALLOC_MAX_FACES = 65536
DM_ERR_TOO_LARGE = -7


class DeltamicError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what} failed: {code} ({_err(code)})")
        self.code = code


class ShapeParams(ctypes.Structure):
    """dm_shape_params (include/deltamic.h)."""
    _fields_ = [("lr", ctypes.c_float), ("lambda_", ctypes.c_float), ("beta1", ctypes.c_float), ("beta2", ctypes.c_float),
                ("eps", ctypes.c_float), ("cg_tol", ctypes.c_float), ("cg_max_iter", ctypes.c_int32), ("solver", ctypes.c_int32)]


class _Grid(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int32 * 3), ("spacing", ctypes.c_float * 3), ("origin", ctypes.c_float * 3)]


_lib = None


def library_path() -> str:
    return _LIB_PATH


def exported_symbols():
    return _SYMBOLS


def load_library():
    """dlopen libdeltamic.so.  Raises (never falls back) when the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2303_10440_b200.build` "
            "(there is no CPU fallback)")
    lib = ctypes.CDLL(_LIB_PATH)
    vp, fp, ip = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p
    lib.dm_plan_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(_Grid), ctypes.c_int, ctypes.c_int32,
                                   ctypes.c_int32, ip, vp]
    lib.dm_plan_set_stream.argtypes = [vp, vp]
    lib.dm_plan_set_slab.argtypes = [vp, ctypes.c_int32, ctypes.c_int32]
    lib.dm_plan_set_option.argtypes = [vp, ctypes.c_int, ctypes.c_double]
    lib.dm_plan_set_face_weights.argtypes = [vp, fp]
    lib.dm_plan_update_face_weights.argtypes = [vp, fp, ctypes.c_int32]
    lib.dm_plan_set_narrow_band.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.c_float]
    lib.dm_mesh_ft_forward.argtypes = [vp, fp, fp]
    lib.dm_mesh_ft_backward.argtypes = [vp, fp, fp, fp]
    lib.dm_mesh_ft_backward_with_spectrum.argtypes = [vp, fp, fp, fp, fp]
    lib.dm_render.argtypes = [vp, fp, ctypes.POINTER(ctypes.c_float), fp]
    lib.dm_render_backward.argtypes = [vp, fp, ctypes.POINTER(ctypes.c_float), fp, fp, ctypes.POINTER(ctypes.c_float)]
    lib.dm_spectrum_to_image.argtypes = [vp, fp, ctypes.POINTER(ctypes.c_float), fp]
    lib.dm_image_to_spectrum_cotangent.argtypes = [vp, fp, ctypes.POINTER(ctypes.c_float), fp]
    lib.dm_plan_stage_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    lib.dm_plan_launch_count.argtypes = [vp]
    lib.dm_plan_launch_count.restype = ctypes.c_int64
    lib.dm_plan_paths_used.argtypes = [vp, ctypes.POINTER(ctypes.c_int32)]
    lib.dm_plan_destroy.argtypes = [vp]
    lib.dm_plan_destroy.restype = None
    lib.dm_error_string.argtypes = [ctypes.c_int]
    lib.dm_error_string.restype = ctypes.c_char_p
    lib.dm_version.restype = ctypes.c_int
    lib.dm_shape_params_default.argtypes = [ctypes.POINTER(ShapeParams)]
    lib.dm_shape_state_create.argtypes = [vp, ctypes.POINTER(ShapeParams), ctypes.POINTER(vp)]
    lib.dm_shape_precondition.argtypes = [vp, vp, fp, fp]
    lib.dm_shape_last_cg_iterations.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_int32)]
    lib.dm_shape_last_cg_residuals.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32)]
    lib.dm_shape_step.argtypes = [vp, vp, fp, fp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_double)]
    lib.dm_shape_state_destroy.argtypes = [vp]
    lib.dm_shape_state_destroy.restype = None
    lib.dm_mesh_ft_forward_noalloc.argtypes = [ctypes.POINTER(_Grid), ctypes.c_int, fp, ip, ctypes.c_int32, fp, vp]
    for name in _SYMBOLS:
        fn = getattr(lib, name)
        if name not in ("dm_plan_launch_count", "dm_plan_destroy", "dm_error_string", "dm_shape_state_destroy"):
            fn.restype = ctypes.c_int
    _lib = lib
    return lib


def _err(code: int) -> str:
    try:
        return load_library().dm_error_string(int(code)).decode()
    except Exception:  # pragma: no cover
        return "?"


def version() -> int:
    return int(load_library().dm_version())


def _check(code: int, what: str):
    if code != 0:
        raise DeltamicError(code, what)


def _cov(psf_cov):
    vals = [float(x) for x in psf_cov]
    if len(vals) != 6:
        raise ValueError("psf_cov must hold 6 numbers: xx, yy, zz, xy, xz, yz")
    return (ctypes.c_float * 6)(*vals)


def mesh_ft_forward_noalloc(n, spacing, mode: int, vertices, faces, out, stream=None):
    """dm_mesh_ft_forward_noalloc: the forward mesh FT for callers that may not allocate device memory (a process whose
    GPU memory is already committed to one arena, a loop that cannot take cudaMalloc's device-wide stall).  No plan; the
    library's scratch is a fixed 4 MiB array inside libdeltamic.so, shared by every call on the GPU, so calls that could
    overlap on one GPU must be serialised by the caller, and ``faces`` may hold at most DM_NOALLOC_MAX_FACES triangles
    (DeltamicError with code DM_ERR_TOO_LARGE beyond that).  Nothing is allocated or converted here either: ``vertices``
    (float32 [n_v, 3]), ``faces`` (int32 [n_f, 3]) and ``out`` (complex64 [n_x, n_y, n_z/2+1], overwritten and returned)
    must already be contiguous CUDA tensors of those types.  Queued on ``stream`` (default: torch's current stream)."""
    import torch

    if not torch.cuda.is_available():
        raise RuntimeError("paper_2303_10440_b200 needs a CUDA device (no CPU fallback)")
    lib = load_library()
    n = tuple(int(v) for v in n)
    for t, dt, name in ((vertices, torch.float32, "vertices"), (faces, torch.int32, "faces"), (out, torch.complex64, "out")):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dt and t.is_contiguous()):
            raise ValueError(f"{name} must be a contiguous CUDA tensor of dtype {dt}")
    if vertices.dim() != 2 or vertices.shape[1] != 3 or faces.dim() != 2 or faces.shape[1] != 3:
        raise ValueError("vertices must be [n_v, 3] and faces [n_f, 3]")
    if tuple(out.shape) != (n[0], n[1], n[2] // 2 + 1):
        raise ValueError("out must have the rfft half-spectrum shape [n_x, n_y, n_z/2+1]")
    grid = _Grid((ctypes.c_int32 * 3)(*n), (ctypes.c_float * 3)(*[float(v) for v in spacing]), (ctypes.c_float * 3)(0.0, 0.0, 0.0))
    s = torch.cuda.current_stream(out.device) if stream is None else stream
    with torch.cuda.device(out.device):
        _check(lib.dm_mesh_ft_forward_noalloc(ctypes.byref(grid), int(mode), vertices.data_ptr(), faces.data_ptr(),
                                              int(faces.shape[0]), out.data_ptr(), ctypes.c_void_p(s.cuda_stream)),
               "dm_mesh_ft_forward_noalloc")
    return out


class Plan:
    """One grid + mode + mesh topology (dm_plan).  Tensors are torch CUDA tensors; all work is queued on
    ``torch.cuda.current_stream()`` at construction time."""

    def __init__(self, n, spacing, origin, mode: int, faces, n_vertices: int, stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2303_10440_b200 needs a CUDA device (no CPU fallback)")
        lib = load_library()
        self._torch = torch
        self.n = tuple(int(v) for v in n)
        self.mode = int(mode)
        self.n_vertices = int(n_vertices)
        faces = faces if isinstance(faces, torch.Tensor) else torch.as_tensor(faces)
        faces = faces.to(device="cuda", dtype=torch.int32).contiguous()
        self.n_faces = int(faces.shape[0])
        self.device = faces.device
        self.stream = torch.cuda.current_stream(self.device) if stream is None else stream
        # bookkeeping for the autograd front end (state_epoch): how often the plan's configuration changed, how many forward
        # spectra it has produced, and whether backward calls take the spectrum of the last render (DM_OPT_REUSE_SPECTRUM)
        self._config_epoch, self._forward_epoch, self._reuse_spectrum = 0, 0, False
        g = _Grid()
        for d in range(3):
            g.n[d] = self.n[d]
            g.spacing[d] = float(spacing[d])
            g.origin[d] = float(origin[d])
        h = ctypes.c_void_p()
        _check(lib.dm_plan_create(ctypes.byref(h), ctypes.byref(g), self.mode, self.n_vertices, self.n_faces,
                                  faces.data_ptr(), self.stream.cuda_stream), "dm_plan_create")
        self._h = h
        self._lib = lib

    # -- helpers ---------------------------------------------------------------------------------------------
    @property
    def spectrum_shape(self):
        return (self.n[0], self.n[1], self.n[2] // 2 + 1)

    def _f32(self, t, numel, name):
        torch = self._torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
            raise ValueError(f"{name} must be a contiguous CUDA tensor")
        if t.dtype == torch.complex64:
            t = torch.view_as_real(t)
        if t.dtype != torch.float32 or t.numel() != numel:
            raise ValueError(f"{name}: expected {numel} float32 values, got {t.numel()} of {t.dtype}")
        return t

    def _vertices(self, v):
        return self._f32(v, self.n_vertices * 3, "vertices")

    def _nk(self):
        return self.n[0] * self.n[1] * (self.n[2] // 2 + 1)

    # -- the C ABI, one method per entry point ------------------------------------------------------------------
    def set_stream(self, stream=None):
        """Queue all later calls on ``stream`` (a torch.cuda.Stream; default: the current stream), e.g. the capturing
        stream of ``torch.cuda.graph``."""
        self.stream = self._torch.cuda.current_stream(self.device) if stream is None else stream
        _check(self._lib.dm_plan_set_stream(self._h, self.stream.cuda_stream), "dm_plan_set_stream")

    def state_epoch(self):
        """A token that changes whenever a later backward call on this plan would differentiate a different function than
        a forward call made now: after set_slab / set_face_weights / set_narrow_band / set_option, and -- only under
        DM_OPT_REUSE_SPECTRUM, where the backward takes F from the last render -- after any other forward, render or shape
        step.  autograd.py compares the token of its forward with the one at backward time."""
        return (self._config_epoch, self._forward_epoch if self._reuse_spectrum else None)

    def set_slab(self, ix_begin: int, ix_end: int):
        self._config_epoch += 1
        _check(self._lib.dm_plan_set_slab(self._h, int(ix_begin), int(ix_end)), "dm_plan_set_slab")

    def set_face_weights(self, weights=None):
        """Per-face density weights (float32 CUDA tensor [n_faces]); ``None`` = all 1."""
        ptr = None if weights is None else self._f32(weights, self.n_faces, "face weights").data_ptr()
        self._config_epoch += 1
        _check(self._lib.dm_plan_set_face_weights(self._h, ptr), "dm_plan_set_face_weights")

    def update_face_weights(self, weights, robust: bool = False):
        """dm_plan_update_face_weights: new weights without the classification pass and its stream synchronisation; the
        caller asserts their class (``robust=False``: one sign, constant per component in volume mode)."""
        ptr = self._f32(weights, self.n_faces, "face weights").data_ptr()
        self._config_epoch += 1
        _check(self._lib.dm_plan_update_face_weights(self._h, ptr, 1 if robust else 0), "dm_plan_update_face_weights")

    def set_narrow_band(self, psf_cov=None, cutoff: float = 0.01):
        """Evaluate only the frequencies with exp(-1/2 k^T B k) > cutoff; ``psf_cov=None`` = off."""
        self._config_epoch += 1
        _check(self._lib.dm_plan_set_narrow_band(self._h, None if psf_cov is None else _cov(psf_cov), float(cutoff)),
               "dm_plan_set_narrow_band")

    def set_option(self, option: int, value: float):
        self._config_epoch += 1
        if int(option) == DM_OPT_REUSE_SPECTRUM:
            self._reuse_spectrum = bool(value)
        _check(self._lib.dm_plan_set_option(self._h, int(option), float(value)), "dm_plan_set_option")

    def mesh_ft_forward(self, vertices, out=None):
        torch = self._torch
        v = self._vertices(vertices)
        if out is None:
            out = torch.zeros(self.spectrum_shape, dtype=torch.complex64, device=self.device)
        o = self._f32(out, 2 * self._nk(), "F")
        self._forward_epoch += 1
        _check(self._lib.dm_mesh_ft_forward(self._h, v.data_ptr(), o.data_ptr()), "dm_mesh_ft_forward")
        return out

    def mesh_ft_backward(self, vertices, dL_dF, out=None, spectrum=None):
        """``spectrum``: the F that mesh_ft_forward returned for these vertices (dm_mesh_ft_backward_with_spectrum)."""
        torch = self._torch
        v = self._vertices(vertices)
        g = self._f32(dL_dF, 2 * self._nk(), "dL_dF")
        if out is None:
            out = torch.empty((self.n_vertices, 3), dtype=torch.float32, device=self.device)
        o = self._f32(out, self.n_vertices * 3, "dL_dvertices")
        if spectrum is not None:
            f = self._f32(spectrum, 2 * self._nk(), "F")
            _check(self._lib.dm_mesh_ft_backward_with_spectrum(self._h, v.data_ptr(), g.data_ptr(), f.data_ptr(),
                                                               o.data_ptr()), "dm_mesh_ft_backward_with_spectrum")
        else:
            _check(self._lib.dm_mesh_ft_backward(self._h, v.data_ptr(), g.data_ptr(), o.data_ptr()), "dm_mesh_ft_backward")
        return out

    def render(self, vertices, psf_cov, out=None):
        torch = self._torch
        v = self._vertices(vertices)
        if out is None:
            out = torch.empty(self.n, dtype=torch.float32, device=self.device)
        o = self._f32(out, self.n[0] * self.n[1] * self.n[2], "image")
        self._forward_epoch += 1
        _check(self._lib.dm_render(self._h, v.data_ptr(), _cov(psf_cov), o.data_ptr()), "dm_render")
        return out

    def render_backward(self, vertices, psf_cov, dL_dimage, out=None, with_psf_grad: bool = False):
        """dL/dvertices; with ``with_psf_grad`` also dL/dSigma (6 floats, host) as a second return value."""
        torch = self._torch
        v = self._vertices(vertices)
        g = self._f32(dL_dimage, self.n[0] * self.n[1] * self.n[2], "dL_dimage")
        if out is None:
            out = torch.empty((self.n_vertices, 3), dtype=torch.float32, device=self.device)
        o = self._f32(out, self.n_vertices * 3, "dL_dvertices")
        dcov = (ctypes.c_float * 6)() if with_psf_grad else None
        _check(self._lib.dm_render_backward(self._h, v.data_ptr(), _cov(psf_cov), g.data_ptr(), o.data_ptr(), dcov),
               "dm_render_backward")
        if with_psf_grad:
            return out, [float(x) for x in dcov]
        return out

    def spectrum_to_image(self, F, psf_cov, out=None):
        torch = self._torch
        f = self._f32(F, 2 * self._nk(), "F")
        if out is None:
            out = torch.empty(self.n, dtype=torch.float32, device=self.device)
        o = self._f32(out, self.n[0] * self.n[1] * self.n[2], "image")
        _check(self._lib.dm_spectrum_to_image(self._h, f.data_ptr(), _cov(psf_cov), o.data_ptr()), "dm_spectrum_to_image")
        return out

    def image_to_spectrum_cotangent(self, dL_dimage, psf_cov, out=None):
        torch = self._torch
        g = self._f32(dL_dimage, self.n[0] * self.n[1] * self.n[2], "dL_dimage")
        if out is None:
            out = torch.empty(self.spectrum_shape, dtype=torch.complex64, device=self.device)
        o = self._f32(out, 2 * self._nk(), "G")
        _check(self._lib.dm_image_to_spectrum_cotangent(self._h, g.data_ptr(), _cov(psf_cov), o.data_ptr()),
               "dm_image_to_spectrum_cotangent")
        return out

    def stage_ms(self):
        ms = (ctypes.c_float * 4)()
        _check(self._lib.dm_plan_stage_ms(self._h, ms), "dm_plan_stage_ms")
        return {"mesh_ft": ms[0], "psf": ms[1], "fft": ms[2], "scatter": ms[3]}

    def launch_count(self) -> int:
        return int(self._lib.dm_plan_launch_count(self._h))

    def paths_used(self):
        """(forward, backward) kernels of the last mesh-FT calls: 0 = fast, 1 = robust, -1 = not called yet."""
        out = (ctypes.c_int32 * 2)()
        _check(self._lib.dm_plan_paths_used(self._h, out), "dm_plan_paths_used")
        return int(out[0]), int(out[1])

    def shape_state(self, **params):
        """A ShapeState (dm_shape_state) of this plan; keyword arguments override dm_shape_params' defaults
        (lr, lambda_, beta1, beta2, eps, cg_tol, cg_max_iter, solver)."""
        return ShapeState(self, **params)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.dm_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass


class ShapeState:
    """Optimiser state of the shape-optimisation step (dm_shape_state).  Argument marshalling only."""

    def __init__(self, plan: Plan, **params):
        self._plan = plan
        self._lib = plan._lib
        prm = ShapeParams()
        _check(self._lib.dm_shape_params_default(ctypes.byref(prm)), "dm_shape_params_default")
        for k, v in params.items():
            if not hasattr(prm, k):
                raise TypeError(f"unknown shape parameter {k}")
            setattr(prm, k, v)
        self.params = prm
        h = ctypes.c_void_p()
        _check(self._lib.dm_shape_state_create(plan._h, ctypes.byref(prm), ctypes.byref(h)), "dm_shape_state_create")
        self._h = h

    def precondition(self, g, out=None):
        """(I + lambda L)^-2 g for a float32 CUDA tensor [n_vertices, 3]."""
        p = self._plan
        gg = p._f32(g, p.n_vertices * 3, "g")
        if out is None:
            out = p._torch.empty((p.n_vertices, 3), dtype=p._torch.float32, device=p.device)
        o = p._f32(out, p.n_vertices * 3, "out")
        _check(self._lib.dm_shape_precondition(p._h, self._h, gg.data_ptr(), o.data_ptr()), "dm_shape_precondition")
        return out

    def last_cg_iterations(self):
        """Iterations of the two solves of the last precondition / step ((-1, -1) for the multi-launch solve)."""
        out = (ctypes.c_int32 * 2)()
        _check(self._lib.dm_shape_last_cg_iterations(self._plan._h, self._h, out), "dm_shape_last_cg_iterations")
        return int(out[0]), int(out[1])

    def last_cg_residuals(self):
        """((rel0, rel1), converged): max-over-columns |r|/|b| the two solves of the last precondition / step stopped at, and
        whether both met cg_tol (False: a solve ran out of cg_max_iter iterations).  Synchronises."""
        rel = (ctypes.c_double * 2)()
        ok = ctypes.c_int32(0)
        _check(self._lib.dm_shape_last_cg_residuals(self._plan._h, self._h, rel, ctypes.byref(ok)), "dm_shape_last_cg_residuals")
        return (float(rel[0]), float(rel[1])), bool(ok.value)

    def step(self, vertices, target, psf_cov, return_loss: bool = False):
        """One step; ``vertices`` is updated in place.  With ``return_loss`` returns Phi_1 before the step (synchronises)."""
        p = self._plan
        v = p._vertices(vertices)
        t = p._f32(target, p.n[0] * p.n[1] * p.n[2], "target")
        loss = ctypes.c_double() if return_loss else None
        p._forward_epoch += 1
        _check(self._lib.dm_shape_step(p._h, self._h, v.data_ptr(), t.data_ptr(), _cov(psf_cov),
                                       ctypes.byref(loss) if return_loss else None), "dm_shape_step")
        return float(loss.value) if return_loss else None

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.dm_shape_state_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass
