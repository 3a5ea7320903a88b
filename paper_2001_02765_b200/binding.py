"""ctypes binding of include/sg_disk.h and include/sg_disk_diag.h -- same names, argument marshalling only.

PyTorch is used for device memory and streams: sigma / Fx / Fy are CUDA float64 tensors whose
``data_ptr()`` is handed to the C ABI, and work is enqueued on torch's current stream.
There is no CPU fallback: a missing library raises at import, a missing GPU raises SgError(SG_ERR_CUDA).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))

SG_OK, SG_ERR_ARG, SG_ERR_LAYOUT, SG_ERR_CUDA, SG_ERR_STATE = 0, -1, -2, -3, -4
_ERR_NAMES = {SG_ERR_ARG: "SG_ERR_ARG", SG_ERR_LAYOUT: "SG_ERR_LAYOUT", SG_ERR_CUDA: "SG_ERR_CUDA",
              SG_ERR_STATE: "SG_ERR_STATE"}

# every symbol include/sg_disk.h and include/sg_disk_diag.h declare (tests check the headers and this list agree)
EXPORTED_SYMBOLS = (
    "sg_create", "sg_destroy", "sg_num_cells", "sg_num_vertices", "sg_layout_info", "sg_cell_geometry",
    "sg_set_density", "sg_set_density_linear", "sg_force", "sg_set_target_range", "sg_set_interaction_mode", "sg_lattice_plan_check", "sg_lattice_plan_fill", "sg_launch_counts", "sg_set_kernel_timing", "sg_get_kernel_times",
    "sg_kernel_model", "sg_kernel_instruction_counts", "sg_measure_fp64_peak", "sg_measure_fp64_mma_peak", "sg_last_error", "sg_version",
    "sg_force_uniform_static", "sg_static_last_error",
)


class SgError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_ERR_NAMES.get(code, code)}: {msg}")
        self.code = code


class _Patch(ctypes.Structure):
    _fields_ = [("level", ctypes.c_int32), ("i0", ctypes.c_int32), ("j0", ctypes.c_int32)]


def lib_path() -> str:
    return os.path.join(HERE, "libsg_disk.so")


_lib = None


def load_library():
    """dlopen libsg_disk.so (built in-tree by paper_2001_02765_b200/build.py).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -m paper_2001_02765_b200.build` "
                          "(or __graft_entry__.build()).  There is no CPU fallback.")
    lib = ctypes.CDLL(path)
    c_i64, c_int, c_dbl, vp = ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_void_p
    dp = ctypes.POINTER(ctypes.c_double)
    lib.sg_create.restype = c_int
    lib.sg_create.argtypes = [ctypes.POINTER(vp), c_int, dp, c_dbl, c_dbl, c_int, ctypes.POINTER(_Patch), c_i64,
                              c_dbl, c_int]
    lib.sg_destroy.restype = None
    lib.sg_destroy.argtypes = [vp]
    lib.sg_num_cells.restype = c_i64
    lib.sg_num_cells.argtypes = [vp]
    lib.sg_num_vertices.restype = c_i64
    lib.sg_num_vertices.argtypes = [vp]
    lib.sg_layout_info.restype = c_int
    lib.sg_layout_info.argtypes = [vp, ctypes.POINTER(c_i64)]
    lib.sg_cell_geometry.restype = c_int
    lib.sg_cell_geometry.argtypes = [vp, dp, dp, dp]
    lib.sg_set_density.restype = c_int
    lib.sg_set_density.argtypes = [vp, vp, vp]
    lib.sg_set_density_linear.restype = c_int
    lib.sg_set_density_linear.argtypes = [vp, vp, vp, vp, vp]
    lib.sg_force.restype = c_int
    lib.sg_force.argtypes = [vp, vp, vp, vp]
    lib.sg_set_target_range.restype = c_int
    lib.sg_set_target_range.argtypes = [vp, c_i64, c_i64]
    lib.sg_set_interaction_mode.restype = c_int
    lib.sg_set_interaction_mode.argtypes = [vp, c_int]
    lib.sg_lattice_plan_check.restype = c_int
    lib.sg_lattice_plan_check.argtypes = [vp, ctypes.POINTER(c_i64)]
    lib.sg_lattice_plan_fill.restype = c_int
    lib.sg_lattice_plan_fill.argtypes = [vp, ctypes.POINTER(c_i64)]
    lib.sg_launch_counts.restype = c_int
    lib.sg_launch_counts.argtypes = [vp, ctypes.POINTER(c_int), ctypes.POINTER(c_int)]
    lib.sg_set_kernel_timing.restype = c_int
    lib.sg_set_kernel_timing.argtypes = [vp, c_int]
    lib.sg_get_kernel_times.restype = c_int
    lib.sg_get_kernel_times.argtypes = [vp, ctypes.POINTER(ctypes.c_float), c_int, ctypes.POINTER(c_int)]
    lib.sg_kernel_model.restype = c_int
    lib.sg_kernel_model.argtypes = [vp, dp, dp, dp, dp]
    lib.sg_kernel_instruction_counts.restype = c_int
    lib.sg_kernel_instruction_counts.argtypes = [c_int, dp, dp]
    lib.sg_measure_fp64_peak.restype = c_int
    lib.sg_measure_fp64_peak.argtypes = [c_int, dp, dp]
    lib.sg_measure_fp64_mma_peak.restype = c_int
    lib.sg_measure_fp64_mma_peak.argtypes = [c_int, dp, dp]
    lib.sg_last_error.restype = ctypes.c_char_p
    lib.sg_last_error.argtypes = [vp]
    lib.sg_version.restype = ctypes.c_char_p
    lib.sg_version.argtypes = []
    lib.sg_force_uniform_static.restype = c_int
    lib.sg_force_uniform_static.argtypes = [c_int, c_int, c_dbl, vp, vp, vp, c_int, vp]
    lib.sg_static_last_error.restype = ctypes.c_char_p
    lib.sg_static_last_error.argtypes = []
    _lib = lib
    return lib


def version() -> str:
    return load_library().sg_version().decode()


def kernel_instruction_counts(kernel: int):
    """(FP64-pipe instructions, FLOPs) per (target, vertex) pair of the direct (0) or slope (1) kernel as built."""
    lib = load_library()
    a, b = ctypes.c_double(), ctypes.c_double()
    rc = lib.sg_kernel_instruction_counts(int(kernel), ctypes.byref(a), ctypes.byref(b))
    if rc != SG_OK:
        raise SgError(rc, "unknown kernel id")
    return a.value, b.value


def measure_fp64_peak(device: int = 0):
    """(FP64 TFLOP/s with FMA = 2, DFMA warp-instructions/s) of a dependent-chain DFMA micro-benchmark."""
    lib = load_library()
    tf, wi = ctypes.c_double(), ctypes.c_double()
    rc = lib.sg_measure_fp64_peak(int(device), ctypes.byref(tf), ctypes.byref(wi))
    if rc != SG_OK:
        raise SgError(rc, lib.sg_last_error(None).decode())
    return tf.value, wi.value


def measure_fp64_mma_peak(device: int = 0):
    """(FP64 TFLOP/s of mma.sync.m8n8k4.f64 alone, total TFLOP/s of DMMA interleaved 1:1 with DFMA)."""
    lib = load_library()
    a, b = ctypes.c_double(), ctypes.c_double()
    rc = lib.sg_measure_fp64_mma_peak(int(device), ctypes.byref(a), ctypes.byref(b))
    if rc != SG_OK:
        raise SgError(rc, lib.sg_last_error(None).decode())
    return a.value, b.value


from .sharding import shard_range  # noqa: E402,F401  (re-exported: one definition of the partition)


def _stream_ptr(device: int):
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream(device).cuda_stream)


STATIC_MAX_VERTICES, STATIC_MAX_SIDE = 66049, 1024     # SG_STATIC_MAX_VERTICES, SG_STATIC_MAX_SIDE of sg_disk_static.h


def force_uniform_static(sigma, G=1.0, Fx=None, Fy=None):
    """sg_force_uniform_static (include/sg_disk_static.h): Fx, Fy of the zeroth-order sum on one uniform grid, for
    callers that cannot let the library allocate device memory (an application arena that owns the GPU, a time-step
    loop that must not take cudaMalloc's device-wide synchronisation, a plug-in under a no-allocation rule).

    sigma: CUDA float64 tensor [ny, nx] (x fastest), at most 256 x 256 cells ((nx+1)*(ny+1) <= 66,049).  Fx, Fy:
    tensors of the same shape to write into; a caller that really cannot allocate passes both (they are created with
    torch.empty only when left out, which is this binding's convenience, not the library's doing).  The library call
    allocates nothing: the vertex weights go to a fixed array inside libsg_disk.so that every call on the device
    shares, so calls that can overlap on the GPU (different streams, no event between them) race; calls on one stream
    are safe.  The first call on a device also looks up that array's address: make it before any stream capture.
    Asynchronous on torch's current stream of sigma's device."""
    import torch
    lib = load_library()
    if not (isinstance(sigma, torch.Tensor) and sigma.is_cuda and sigma.dtype == torch.float64 and sigma.dim() == 2
            and sigma.is_contiguous()):
        raise SgError(SG_ERR_ARG, "sigma must be a contiguous CUDA float64 tensor [ny, nx]")
    ny, nx = sigma.shape
    dev = sigma.device.index
    if Fx is None:
        Fx = torch.empty_like(sigma)
    if Fy is None:
        Fy = torch.empty_like(sigma)
    for t, name in ((Fx, "Fx"), (Fy, "Fy")):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and t.shape == sigma.shape and t.device == sigma.device):
            raise SgError(SG_ERR_ARG, f"{name} must be a contiguous CUDA float64 tensor shaped like sigma, on its device")
    rc = lib.sg_force_uniform_static(int(nx), int(ny), float(G), ctypes.c_void_p(sigma.data_ptr()),
                                     ctypes.c_void_p(Fx.data_ptr()), ctypes.c_void_p(Fy.data_ptr()), int(dev),
                                     _stream_ptr(dev))
    if rc != SG_OK:
        raise SgError(rc, lib.sg_static_last_error().decode())
    return Fx, Fy


class SgDisk:
    """One AMR layout on one GPU: sg_create / sg_set_density / sg_force / sg_destroy."""

    def __init__(self, n_levels, cell_width, x0, y0, patch_cells, patches, G=1.0, device=0):
        self._lib = load_library()
        self._ctx = ctypes.c_void_p()
        cw = np.ascontiguousarray(cell_width, dtype=np.float64)
        pa = np.ascontiguousarray(patches, dtype=np.int32).reshape(-1, 3)
        self.device = int(device)
        rc = self._lib.sg_create(ctypes.byref(self._ctx), int(n_levels),
                                 cw.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), float(x0), float(y0),
                                 int(patch_cells), pa.ctypes.data_as(ctypes.POINTER(_Patch)), pa.shape[0],
                                 float(G), self.device)
        if rc != SG_OK:
            self._ctx = ctypes.c_void_p()
            raise SgError(rc, self._lib.sg_last_error(None).decode())
        self._first, self._count = 0, self.num_cells

    @classmethod
    def from_layout(cls, lay, G=1.0, device=0):
        """From a workloads.Layout-like object (n_levels, cell_width, x0, y0, P, patches)."""
        return cls(lay.n_levels, lay.cell_width, lay.x0, lay.y0, lay.P, lay.patches, G=G, device=device)

    # -- bookkeeping ---------------------------------------------------------------------------
    def _check(self, rc):
        if rc != SG_OK:
            raise SgError(rc, self._lib.sg_last_error(self._ctx).decode())

    def close(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            self._lib.sg_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    @property
    def num_cells(self) -> int:
        return int(self._lib.sg_num_cells(self._ctx))

    @property
    def num_vertices(self) -> int:
        return int(self._lib.sg_num_vertices(self._ctx))

    def layout_info(self) -> dict:
        a = (ctypes.c_int64 * 8)()
        self._check(self._lib.sg_layout_info(self._ctx, a))
        keys = ("n_cells", "n_vertices", "n_vertex_x", "n_vertex_y", "n_target_x", "n_target_y", "balanced",
                "device_bytes")
        return dict(zip(keys, [int(v) for v in a]))

    def cell_geometry(self):
        n = self.num_cells
        xc, yc, h = np.empty(n), np.empty(n), np.empty(n)
        dp = ctypes.POINTER(ctypes.c_double)
        self._check(self._lib.sg_cell_geometry(self._ctx, xc.ctypes.data_as(dp), yc.ctypes.data_as(dp),
                                               h.ctypes.data_as(dp)))
        return xc, yc, h

    # -- the hot path --------------------------------------------------------------------------
    def set_density(self, sigma):
        """sigma: CUDA float64 tensor [N] in library cell order (asynchronous on the current stream)."""
        self._require_cuda(sigma, self.num_cells, "sigma")
        self._check(self._lib.sg_set_density(self._ctx, ctypes.c_void_p(sigma.data_ptr()), _stream_ptr(self.device)))

    def set_density_linear(self, sigma, dx, dy):
        """sigma, dx, dy: CUDA float64 tensors [N] (value and physical slopes of Eq. 6 per leaf); the next
        force() calls include the slope terms."""
        for t, name in ((sigma, "sigma"), (dx, "dx"), (dy, "dy")):
            self._require_cuda(t, self.num_cells, name)
        self._check(self._lib.sg_set_density_linear(self._ctx, ctypes.c_void_p(sigma.data_ptr()),
                                                    ctypes.c_void_p(dx.data_ptr()), ctypes.c_void_p(dy.data_ptr()),
                                                    _stream_ptr(self.device)))

    def set_target_range(self, first: int, count: int):
        self._check(self._lib.sg_set_target_range(self._ctx, int(first), int(count)))
        self._first, self._count = int(first), int(count)

    def set_interaction_mode(self, mode: str):
        """'direct' (every pair: sqrt + 2 ln), 'lattice' (per-patch-pair offset tables; P = 8 or 16) or
        'lattice_blocked' (the register-blocked offset-table kernels at any size; P = 16)."""
        self._check(self._lib.sg_set_interaction_mode(self._ctx, {"direct": 0, "lattice": 1, "lattice_blocked": 2, "lattice_incta": 3}[mode]))

    def lattice_plan_check(self):
        """Host-side replay of the lattice-mode launch plan (see sg_lattice_plan_check)."""
        out = (ctypes.c_int64 * 16)()
        self._check(self._lib.sg_lattice_plan_check(self._ctx, out))
        v = list(out)
        return {"pairs_per_class": v[0:5], "duplicates": v[5], "wrong_level": v[6], "groups": v[7:10],
                "offsets": v[10], "available": bool(v[11]), "patches_missing_from_launched_lists": v[12]}

    def lattice_plan_fill(self):
        """Per pair class: offsets visited, offsets with a source patch for some target of the group, patch pairs."""
        out = (ctypes.c_int64 * 15)()
        self._check(self._lib.sg_lattice_plan_fill(self._ctx, out))
        v = list(out)
        return [dict(offsets=v[3 * k], live_offsets=v[3 * k + 1], pairs=v[3 * k + 2]) for k in range(5)]

    def force(self, Fx=None, Fy=None):
        """Fx, Fy (CUDA float64 [count]) at the leaf centres of the current target range."""
        import torch
        dev = torch.device("cuda", self.device)
        if Fx is None:
            Fx = torch.empty(self._count, dtype=torch.float64, device=dev)
        if Fy is None:
            Fy = torch.empty(self._count, dtype=torch.float64, device=dev)
        self._require_cuda(Fx, self._count, "Fx")
        self._require_cuda(Fy, self._count, "Fy")
        self._check(self._lib.sg_force(self._ctx, ctypes.c_void_p(Fx.data_ptr()), ctypes.c_void_p(Fy.data_ptr()),
                                       _stream_ptr(self.device)))
        return Fx, Fy

    def launch_counts(self):
        a, b = ctypes.c_int(), ctypes.c_int()
        self._check(self._lib.sg_launch_counts(self._ctx, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def set_kernel_timing(self, enable: bool = True):
        self._check(self._lib.sg_set_kernel_timing(self._ctx, int(bool(enable))))

    def kernel_times_ms(self):
        """Interaction-kernel durations (ms) of the force() calls since set_kernel_timing(True), oldest first."""
        buf, n = (ctypes.c_float * 64)(), ctypes.c_int()
        self._check(self._lib.sg_get_kernel_times(self._ctx, buf, 64, ctypes.byref(n)))
        return [float(buf[i]) for i in range(n.value)]

    def kernel_model(self) -> dict:
        a, b, c, e = ctypes.c_double(), ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        self._check(self._lib.sg_kernel_model(self._ctx, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c),
                                              ctypes.byref(e)))
        return dict(fp64_instr_per_pair=a.value, flops_per_pair=b.value, pair_evaluations=c.value,
                    executed_evaluations=e.value)

    def _require_cuda(self, t, n, name):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and t.numel() == n and t.device.index == self.device):
            raise SgError(SG_ERR_ARG, f"{name} must be a contiguous CUDA float64 tensor of {n} elements on "
                                      f"cuda:{self.device}")
