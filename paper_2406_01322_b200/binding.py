"""ctypes binding of include/psdns.h.  Same names as the C ABI; torch supplies device memory
and the stream.  No arithmetic happens here."""
from __future__ import annotations

import ctypes as C
import os

PHYSICAL, SPECTRAL = 0, 1
_HERE = os.path.dirname(os.path.abspath(__file__))

EXPORTS = [
    "psdns_workspace_bytes", "psdns_init", "psdns_set_state", "psdns_step", "psdns_get_state",
    "psdns_transform_roundtrip", "psdns_run_host", "psdns_run_host_wait", "psdns_launch_count", "psdns_kernel_timing",
    "psdns_kernel_time_ms", "psdns_destroy", "psdns_last_error",
    "psdns_history_bytes", "psdns_get_history", "psdns_set_history",
    "psdns_set_option", "psdns_get_info", "psdns_workspace_bytes_unfused", "psdns_diagnostics",
    "psdns_render_isosurface", "psdns_measure_fp64_peak", "psdns_diagnostics_static",
]

STATIC_SCRATCH_DOUBLES = 2048   # PSDNS_STATIC_SCRATCH_DOUBLES of include/psdns.h


class PsdnsError(RuntimeError):
    pass


class psdns_grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("lx", C.c_double), ("ly", C.c_double)]


class psdns_camera(C.Structure):
    _fields_ = [("eye", C.c_double * 3), ("target", C.c_double * 3), ("up", C.c_double * 3), ("fov_y_deg", C.c_double),
                ("width", C.c_int), ("height", C.c_int), ("step", C.c_double), ("light", C.c_double * 3)]


class psdns_params(C.Structure):
    _fields_ = [("re", C.c_double), ("pe", C.c_double), ("ch", C.c_double), ("we", C.c_double),
                ("dt", C.c_double), ("gradp_x", C.c_double), ("visc_ratio", C.c_double),
                ("phase_field", C.c_int), ("dealias", C.c_int), ("wall_top", C.c_int), ("wall_bottom", C.c_int),
                ("surface_tension_form", C.c_int), ("convection_form", C.c_int)]


def lib_path() -> str:
    return os.path.join(_HERE, "libpsdns.so")


_lib = None


def load_library():
    """dlopen libpsdns.so (built in-tree by `python -m paper_2406_01322_b200.build` or
    `__graft_entry__.build()`).  Fails loudly if it is missing - there is no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise PsdnsError(f"{path} not found: build it with `python -m paper_2406_01322_b200.build`")
    lib = C.CDLL(path)
    vp, ci, cd = C.c_void_p, C.c_int, C.c_double
    lib.psdns_workspace_bytes.restype = C.c_size_t
    lib.psdns_workspace_bytes.argtypes = [C.POINTER(psdns_grid), C.POINTER(psdns_params)]
    lib.psdns_init.restype = ci
    lib.psdns_init.argtypes = [C.POINTER(psdns_grid), C.POINTER(psdns_params), vp, C.c_size_t, vp, C.POINTER(vp)]
    lib.psdns_set_state.restype = ci
    lib.psdns_set_state.argtypes = [vp, ci, vp, vp, vp, vp]
    lib.psdns_step.restype = ci
    lib.psdns_step.argtypes = [vp, ci]
    lib.psdns_get_state.restype = ci
    lib.psdns_get_state.argtypes = [vp, ci, vp, vp, vp, vp]
    lib.psdns_transform_roundtrip.restype = ci
    lib.psdns_transform_roundtrip.argtypes = [vp, ci, vp, vp, vp]
    lib.psdns_run_host.restype = ci
    lib.psdns_run_host.argtypes = [vp, ci, ci] + [vp] * 8
    lib.psdns_run_host_wait.restype = ci
    lib.psdns_run_host_wait.argtypes = [vp]
    lib.psdns_launch_count.restype = C.c_longlong
    lib.psdns_launch_count.argtypes = [vp]
    lib.psdns_kernel_timing.restype = ci
    lib.psdns_kernel_timing.argtypes = [vp, C.c_char_p, ci]
    lib.psdns_kernel_time_ms.restype = ci
    lib.psdns_kernel_time_ms.argtypes = [vp, C.POINTER(cd), C.POINTER(C.c_longlong)]
    lib.psdns_history_bytes.restype = C.c_size_t
    lib.psdns_history_bytes.argtypes = [vp]
    lib.psdns_get_history.restype = ci
    lib.psdns_get_history.argtypes = [vp, vp, C.c_size_t]
    lib.psdns_set_history.restype = ci
    lib.psdns_set_history.argtypes = [vp, vp, C.c_size_t]
    lib.psdns_diagnostics.restype = ci
    lib.psdns_diagnostics.argtypes = [vp, vp]
    lib.psdns_diagnostics_static.restype = ci
    lib.psdns_diagnostics_static.argtypes = [vp, vp]
    lib.psdns_render_isosurface.restype = ci
    lib.psdns_render_isosurface.argtypes = [vp, C.POINTER(psdns_camera), cd, vp, vp, vp]
    lib.psdns_measure_fp64_peak.restype = ci
    lib.psdns_measure_fp64_peak.argtypes = [vp, C.POINTER(cd)]
    lib.psdns_set_option.restype = ci
    lib.psdns_set_option.argtypes = [vp, C.c_char_p, cd]
    lib.psdns_get_info.restype = cd
    lib.psdns_get_info.argtypes = [vp, C.c_char_p]
    lib.psdns_workspace_bytes_unfused.restype = C.c_size_t
    lib.psdns_workspace_bytes_unfused.argtypes = [C.POINTER(psdns_grid), C.POINTER(psdns_params)]
    lib.psdns_destroy.restype = ci
    lib.psdns_destroy.argtypes = [vp]
    lib.psdns_last_error.restype = C.c_char_p
    lib.psdns_last_error.argtypes = [vp]
    _lib = lib
    return lib


def exported_symbols():
    lib = load_library()
    return {name: hasattr(lib, name) for name in EXPORTS}


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


class Solver:
    """Thin owner of a psdns handle.  Fields are torch CUDA tensors in the boundary layouts of
    include/psdns.h: PHYSICAL float64 [nz, ny, nx]; SPECTRAL complex128 [nz, ny, nx//2+1]."""

    def __init__(self, nx, ny, nz, lx, ly, *, re, dt, pe=1.0, ch=1.0, we=1.0, gradp_x=0.0,
                 visc_ratio=1.0, phase_field=1, dealias=1, device="cuda:0", unfused_workspace=False,
                 wall_top=0, wall_bottom=0, surface_tension_form=0, convection_form=0):
        import torch
        self.torch = torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise PsdnsError("libpsdns needs a CUDA device (no CPU fallback)")
        self.device = torch.device(device)
        self.grid = psdns_grid(nx, ny, nz, lx, ly)
        self.params = psdns_params(re, pe, ch, we, dt, gradp_x, visc_ratio, phase_field, dealias, wall_top, wall_bottom,
                                   surface_tension_form, convection_form)
        self.nx, self.ny, self.nz = nx, ny, nz
        self.phase = bool(phase_field)
        wsfn = self.lib.psdns_workspace_bytes_unfused if unfused_workspace else self.lib.psdns_workspace_bytes
        nbytes = wsfn(C.byref(self.grid), C.byref(self.params))
        if nbytes == 0:
            raise PsdnsError("psdns_workspace_bytes: invalid grid/params")
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = torch.cuda.current_stream(self.device)
            self.handle = C.c_void_p()
            rc = self.lib.psdns_init(C.byref(self.grid), C.byref(self.params), C.c_void_p(self.workspace.data_ptr()),
                                     nbytes, C.c_void_p(self.stream.cuda_stream), C.byref(self.handle))
        self._check(rc)

    # -- helpers --
    def _check(self, rc):
        if rc != 0:
            msg = self.lib.psdns_last_error(self.handle) if self.handle else b""
            raise PsdnsError(f"libpsdns error {rc}: {msg.decode() if msg else ''}")

    def _shape(self, space):
        if space == PHYSICAL:
            return (self.nz, self.ny, self.nx), self.torch.float64
        return (self.nz, self.ny, self.nx // 2 + 1), self.torch.complex128

    def _chk_field(self, t, space):
        shape, dt = self._shape(space)
        if t is None:
            return
        if tuple(t.shape) != shape or t.dtype != dt or not t.is_cuda or not t.is_contiguous():
            raise PsdnsError(f"field must be a contiguous CUDA tensor {shape} {dt}")

    def empty_fields(self, space):
        shape, dt = self._shape(space)
        n = 4 if self.phase else 3
        return [self.torch.empty(shape, dtype=dt, device=self.device) for _ in range(n)]

    # -- C ABI calls --
    def set_state(self, space, u, v, w, phi=None):
        for t in (u, v, w, phi):
            self._chk_field(t, space)
        self._check(self.lib.psdns_set_state(self.handle, space, _ptr(u), _ptr(v), _ptr(w), _ptr(phi)))

    def step(self, nsteps=1):
        self._check(self.lib.psdns_step(self.handle, nsteps))

    def get_state(self, space):
        out = self.empty_fields(space)
        phi = out[3] if self.phase else None
        self._check(self.lib.psdns_get_state(self.handle, space, _ptr(out[0]), _ptr(out[1]), _ptr(out[2]), _ptr(phi)))
        return out

    def transform_roundtrip(self, start_space, x, want_mid=False):
        self._chk_field(x, start_space)
        shape, dt = self._shape(start_space)
        out = self.torch.empty(shape, dtype=dt, device=self.device)
        mid = None
        if want_mid:
            mshape, mdt = self._shape(1 - start_space)
            mid = self.torch.empty(mshape, dtype=mdt, device=self.device)
        self._check(self.lib.psdns_transform_roundtrip(self.handle, start_space, _ptr(x), _ptr(out), _ptr(mid)))
        return (out, mid) if want_mid else out

    def run_host(self, space, nsteps, h_in, h_out):
        """h_in / h_out: lists of pinned host tensors (boundary layout).  Asynchronous: h_out is valid after run_host_wait()."""
        pi = [C.c_void_p(t.data_ptr()) if t is not None else None for t in (list(h_in) + [None] * 4)[:4]]
        po = [C.c_void_p(t.data_ptr()) if t is not None else None for t in (list(h_out) + [None] * 4)[:4]]
        self._check(self.lib.psdns_run_host(self.handle, space, nsteps, *pi, *po))

    def run_host_wait(self):
        """Blocks until the device -> host copies of the last run_host have landed in h_out."""
        self._check(self.lib.psdns_run_host_wait(self.handle))

    def get_history(self):
        """Opaque device blob with the hidden state of the time integration (exact restart)."""
        n = int(self.lib.psdns_history_bytes(self.handle))
        blob = self.torch.empty(n, dtype=self.torch.uint8, device=self.device)
        self._check(self.lib.psdns_get_history(self.handle, _ptr(blob), n))
        return blob

    def set_history(self, blob):
        self._check(self.lib.psdns_set_history(self.handle, _ptr(blob), blob.numel()))

    def launch_count(self):
        return int(self.lib.psdns_launch_count(self.handle))

    def kernel_timing(self, name, enable=True):
        self._check(self.lib.psdns_kernel_timing(self.handle, name.encode(), 1 if enable else 0))

    def kernel_time_ms(self):
        ms, n = C.c_double(), C.c_longlong()
        self._check(self.lib.psdns_kernel_time_ms(self.handle, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    DIAG_NAMES = ("mean_phi", "max_div", "kinetic_energy", "shear_top", "shear_bottom", "bulk_velocity")

    def diagnostics(self):
        """psdns_diagnostics into a fresh device tensor of 8 doubles (asynchronous; index with DIAG_NAMES order)."""
        out = self.torch.empty(8, dtype=self.torch.float64, device=self.device)
        self._check(self.lib.psdns_diagnostics(self.handle, _ptr(out)))
        return out

    def diagnostics_static(self, out):
        """psdns_diagnostics_static into the caller's device tensor `out` (8 doubles): no allocation on either side of the
        boundary; the reduction partials live in the library's file-scope device array (include/psdns.h)."""
        if out.dtype != self.torch.float64 or out.numel() != 8 or not out.is_cuda or not out.is_contiguous():
            raise PsdnsError("diagnostics_static: out must be a contiguous CUDA tensor of 8 doubles")
        self._check(self.lib.psdns_diagnostics_static(self.handle, _ptr(out)))
        return out

    def render_isosurface(self, eye, target, up=(0.0, 0.0, 1.0), fov_y_deg=40.0, width=64, height=48, step=0.02,
                          light=(0.3, -0.5, 0.8), iso=0.0, field=None):
        """psdns_render_isosurface: (intensity, depth) device tensors [height, width]; field = None renders the state's phi."""
        if field is not None:
            self._chk_field(field, PHYSICAL)
        v3 = C.c_double * 3
        cam = psdns_camera(v3(*eye), v3(*target), v3(*up), fov_y_deg, width, height, step, v3(*light))
        inten = self.torch.empty((height, width), dtype=self.torch.float64, device=self.device)
        depth = self.torch.empty((height, width), dtype=self.torch.float64, device=self.device)
        self._check(self.lib.psdns_render_isosurface(self.handle, C.byref(cam), float(iso), _ptr(field), _ptr(inten), _ptr(depth)))
        return inten, depth

    def measure_fp64_peak(self):
        """FP64 FMA-chain microbenchmark, TFLOP/s (synchronises the stream)."""
        tf = C.c_double()
        self._check(self.lib.psdns_measure_fp64_peak(self.handle, C.byref(tf)))
        return tf.value

    def set_option(self, name, value):
        self._check(self.lib.psdns_set_option(self.handle, name.encode(), float(value)))

    def get_info(self, name):
        return float(self.lib.psdns_get_info(self.handle, name.encode()))

    def close(self):
        if getattr(self, "handle", None):
            self.lib.psdns_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
