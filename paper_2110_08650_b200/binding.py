"""Thin ctypes binding of libpic_b200.so (include/pic_b200.h) — argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; torch is used for device
memory (the workspace and the caller's arrays) and for the stream.  There is no CPU
fallback: if the library cannot be loaded, or no CUDA device is present when a context
is created, this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence, Tuple

import torch

from .build import LIB, build_library

PIC_OK, PIC_EINVAL, PIC_ENOMEM, PIC_ECUDA, PIC_ESTATE, PIC_EDEVICE = 0, -1, -2, -3, -4, -5
_CODES = {0: "PIC_OK", -1: "PIC_EINVAL", -2: "PIC_ENOMEM", -3: "PIC_ECUDA", -4: "PIC_ESTATE", -5: "PIC_EDEVICE"}

# every symbol include/pic_b200.h declares
SYMBOLS = (
    "pic_workspace_bytes", "pic_create", "pic_set_species", "pic_load_particles", "pic_set_fields",
    "pic_step", "pic_get_current", "pic_get_particles", "pic_get_counts", "pic_get_stats", "pic_sync",
    "pic_set_option", "pic_get_timing", "pic_launch_count", "pic_last_error", "pic_destroy",
    "pic_update_fields", "pic_get_fields", "pic_deposit_current_noalloc", "pic_set_current",
)


class PicError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_CODES.get(code, code)}: {msg}")
        self.code = code


_lib = None


def load_library(build_if_missing: bool = True) -> C.CDLL:
    """dlopen libpic_b200.so (building it with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = LIB
    if build_if_missing:
        path = build_library()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it with `python -m paper_2110_08650_b200.build` "
                           "(the product has no CPU fallback)")
    L = C.CDLL(path)
    vp, i32, i64, u64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64
    L.pic_workspace_bytes.argtypes = [C.POINTER(i32), C.POINTER(i32), i32, i64, C.POINTER(u64)]
    L.pic_create.argtypes = [C.POINTER(vp), C.POINTER(i32), C.POINTER(C.c_double), C.c_double,
                             C.POINTER(i32), i32, i64, vp, u64, vp]
    L.pic_set_species.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.pic_load_particles.argtypes = [vp, i64] + [vp] * 8
    L.pic_set_fields.argtypes = [vp] + [vp] * 6
    L.pic_step.argtypes = [vp, i32]
    L.pic_get_current.argtypes = [vp] + [vp] * 3
    L.pic_get_particles.argtypes = [vp, i64, C.POINTER(i64)] + [vp] * 10
    L.pic_get_counts.argtypes = [vp, vp]
    L.pic_get_stats.argtypes = [vp, C.POINTER(i64)]
    L.pic_sync.argtypes = [vp]
    L.pic_set_option.argtypes = [vp, C.c_char_p, i64]
    L.pic_get_timing.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(i64)]
    L.pic_launch_count.argtypes = [vp]
    L.pic_launch_count.restype = i64
    L.pic_last_error.argtypes = [vp]
    L.pic_last_error.restype = C.c_char_p
    L.pic_destroy.argtypes = [vp]
    L.pic_update_fields.argtypes = [vp]
    L.pic_get_fields.argtypes = [vp] + [vp] * 6
    for name in SYMBOLS:
        if name not in ("pic_launch_count", "pic_last_error"):
            getattr(L, name).restype = i32
    _lib = L
    return L


def _ptr(t: Optional[torch.Tensor], dtype: torch.dtype, n: Optional[int] = None, what: str = "array"):
    if t is None:
        return None
    if not t.is_cuda:
        raise ValueError(f"{what}: expected a CUDA tensor (no CPU path exists)")
    if t.dtype != dtype:
        raise TypeError(f"{what}: expected {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{what}: tensor must be contiguous")
    if n is not None and t.numel() != n:
        raise ValueError(f"{what}: expected {n} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


def workspace_bytes(grid: Sequence[int], supercell: Sequence[int], shape_order: int, max_particles: int) -> int:
    L = load_library()
    out = C.c_uint64(0)
    rc = L.pic_workspace_bytes((C.c_int32 * 3)(*grid), (C.c_int32 * 3)(*supercell), int(shape_order),
                               int(max_particles), C.byref(out))
    if rc != PIC_OK:
        raise PicError(rc, L.pic_last_error(None).decode())
    return int(out.value)


class Pic:
    """One simulation context.  Method names mirror the C ABI without the ``pic_`` prefix."""

    def __init__(self, grid, cell=(1.0, 1.0, 1.0), dt=0.5, supercell=(8, 8, 4), shape_order=1,
                 max_particles=0, device="cuda:0", stream: Optional[torch.cuda.Stream] = None,
                 workspace: Optional[torch.Tensor] = None):
        self._L = load_library()
        self._h = C.c_void_p(None)
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2110_08650_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.device = torch.device(device)
        self.grid = tuple(int(v) for v in grid)
        self.cell = tuple(float(v) for v in cell)
        self.supercell = tuple(int(v) for v in supercell)
        self.shape_order = int(shape_order)
        self.dt = float(dt)
        self.max_particles = int(max_particles)
        self.n_supercells = 1
        for a in range(3):
            self.n_supercells *= self.grid[a] // max(self.supercell[a], 1)
        nbytes = workspace_bytes(self.grid, self.supercell, self.shape_order, self.max_particles)
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            if workspace is not None:
                if not workspace.is_cuda or workspace.dtype != torch.uint8 or workspace.numel() < nbytes + 256:
                    raise ValueError("workspace must be a CUDA uint8 tensor of >= workspace_bytes()+256 elements")
                self.workspace = workspace
            else:
                self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        aligned = (base + 255) // 256 * 256
        h = C.c_void_p(None)
        rc = self._L.pic_create(C.byref(h), (C.c_int32 * 3)(*self.grid), (C.c_double * 3)(*self.cell), self.dt,
                                (C.c_int32 * 3)(*self.supercell), self.shape_order, self.max_particles,
                                C.c_void_p(aligned), nbytes, C.c_void_p(self.stream.cuda_stream))
        if rc != PIC_OK:
            raise PicError(rc, self._L.pic_last_error(None).decode())
        self._h = h
        self.workspace_nbytes = nbytes

    # -- helpers
    def _check(self, rc: int):
        if rc != PIC_OK:
            raise PicError(rc, self._L.pic_last_error(self._h).decode())

    @property
    def n_cells(self) -> int:
        return self.grid[0] * self.grid[1] * self.grid[2]

    # -- the C ABI
    def set_species(self, q: Sequence[float], m: Sequence[float]):
        n = len(q)
        self._check(self._L.pic_set_species(self._h, n, (C.c_double * n)(*q), (C.c_double * n)(*m)))

    def load_particles(self, x, y, z, ux, uy, uz, w, species=None):
        n = int(x.numel())
        f64, f32 = torch.float64, torch.float32
        args = [_ptr(x, f64, n, "x"), _ptr(y, f64, n, "y"), _ptr(z, f64, n, "z"),
                _ptr(ux, f32, n, "ux"), _ptr(uy, f32, n, "uy"), _ptr(uz, f32, n, "uz"),
                _ptr(w, f32, n, "w"), _ptr(species, torch.int32, n, "species")]
        self._check(self._L.pic_load_particles(self._h, n, *args))

    def set_fields(self, fields6: torch.Tensor):
        """fields6: float32 CUDA tensor [6, nz, ny, nx] (Ex,Ey,Ez,Bx,By,Bz at their Yee locations)."""
        _ptr(fields6, torch.float32, 6 * self.n_cells, "fields")
        nb = self.n_cells * 4
        base = fields6.data_ptr()
        self._check(self._L.pic_set_fields(self._h, *[C.c_void_p(base + c * nb) for c in range(6)]))

    def step(self, n: int = 1):
        self._check(self._L.pic_step(self._h, int(n)))

    def update_fields(self):
        """One Yee update of E, B with the last step's J (pic_update_fields)."""
        self._check(self._L.pic_update_fields(self._h))

    def get_fields(self) -> torch.Tensor:
        """float32 [6, nz, ny, nx]: the current Ex,Ey,Ez,Bx,By,Bz."""
        nx, ny, nz = self.grid
        F = torch.empty((6, nz, ny, nx), dtype=torch.float32, device=self.device)
        nb = self.n_cells * 4
        self._check(self._L.pic_get_fields(self._h, *[C.c_void_p(F.data_ptr() + c * nb) for c in range(6)]))
        return F

    def set_current(self, J: torch.Tensor):
        """J: float32 [3, nz, ny, nx] on the device: the current the next update_fields uses (pic_set_current)."""
        nx, ny, nz = self.grid
        if tuple(J.shape) != (3, nz, ny, nx) or J.dtype != torch.float32 or not J.is_cuda or not J.is_contiguous():
            raise ValueError("J: expected a contiguous CUDA float32 tensor of shape [3, nz, ny, nx]")
        nb = self.n_cells * 4
        self._check(self._L.pic_set_current(self._h, *[C.c_void_p(J.data_ptr() + c * nb) for c in range(3)]))

    def get_current(self) -> torch.Tensor:
        """float32 [3, nz, ny, nx]: J of the last step."""
        nx, ny, nz = self.grid
        J = torch.empty((3, nz, ny, nx), dtype=torch.float32, device=self.device)
        nb = self.n_cells * 4
        self._check(self._L.pic_get_current(self._h, *[C.c_void_p(J.data_ptr() + c * nb) for c in range(3)]))
        return J

    def get_particles(self, capacity: Optional[int] = None) -> dict:
        cap = int(capacity if capacity is not None else self.max_particles)
        dev = self.device
        out = dict(
            x=torch.empty(cap, dtype=torch.float64, device=dev), y=torch.empty(cap, dtype=torch.float64, device=dev),
            z=torch.empty(cap, dtype=torch.float64, device=dev), ux=torch.empty(cap, dtype=torch.float32, device=dev),
            uy=torch.empty(cap, dtype=torch.float32, device=dev), uz=torch.empty(cap, dtype=torch.float32, device=dev),
            w=torch.empty(cap, dtype=torch.float32, device=dev), species=torch.empty(cap, dtype=torch.int32, device=dev),
            id=torch.empty(cap, dtype=torch.int32, device=dev), supercell=torch.empty(cap, dtype=torch.int32, device=dev))
        n = C.c_int64(0)
        self._check(self._L.pic_get_particles(
            self._h, cap, C.byref(n), *[C.c_void_p(out[k].data_ptr()) for k in
                                        ("x", "y", "z", "ux", "uy", "uz", "w", "species", "id", "supercell")]))
        return {k: v[: n.value] for k, v in out.items()}

    def get_counts(self) -> torch.Tensor:
        c = torch.empty(self.n_supercells, dtype=torch.int32, device=self.device)
        self._check(self._L.pic_get_counts(self._h, C.c_void_p(c.data_ptr())))
        return c

    def get_stats(self, check: bool = True) -> dict:
        s = (C.c_int64 * 8)()
        rc = self._L.pic_get_stats(self._h, s)
        if check:
            self._check(rc)
        keys = ("particles", "leavers_last", "frames_used", "frames_pool", "max_count", "steps", "leavers_cum", "error")
        return dict(zip(keys, (int(v) for v in s)))

    def sync(self):
        self._check(self._L.pic_sync(self._h))

    def set_option(self, key: str, value: int):
        self._check(self._L.pic_set_option(self._h, key.encode(), int(value)))

    def get_timing(self) -> Tuple[float, int]:
        """(total ms of step-kernel launches since the last call, number of launches); needs option timing=1."""
        ms, n = C.c_double(0.0), C.c_int64(0)
        self._check(self._L.pic_get_timing(self._h, C.byref(ms), C.byref(n)))
        return float(ms.value), int(n.value)

    def launch_count(self) -> int:
        return int(self._L.pic_launch_count(self._h))

    def destroy(self):
        if self._h:
            self._L.pic_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


NOALLOC_MAX_CELLS = 262144     # PIC_NOALLOC_MAX_CELLS of include/pic_b200.h


def deposit_current_noalloc(grid: Sequence[int], cell: Sequence[float], dt: float, shape_order: int,
                            x0: torch.Tensor, y0: torch.Tensor, z0: torch.Tensor,
                            x1: torch.Tensor, y1: torch.Tensor, z1: torch.Tensor, qw: torch.Tensor,
                            out: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """pic_deposit_current_noalloc (include/pic_b200.h): the Esirkepov current of particles that moved x0 -> x1, into
    the CALLER's `out` ([3, nz, ny, nx] float32, overwritten).  Marshalling only; nothing is allocated on the device,
    here or in the library (scratch is a fixed 6 MiB device array: at most NOALLOC_MAX_CELLS cells).  Calls that
    overlap on the GPU share that scratch and race: keep them on one stream."""
    L = load_library()
    n = int(x0.numel())
    nx, ny, nz = (int(v) for v in grid)
    if tuple(out.shape) != (3, nz, ny, nx) or out.dtype != torch.float32 or not out.is_cuda or not out.is_contiguous():
        raise ValueError("out: expected a contiguous CUDA float32 tensor of shape [3, nz, ny, nx]")
    args = [_ptr(t, torch.float64, n, k) for k, t in (("x0", x0), ("y0", y0), ("z0", z0), ("x1", x1), ("y1", y1), ("z1", z1))]
    args.append(_ptr(qw, torch.float32, n, "qw"))
    st = stream if stream is not None else torch.cuda.current_stream(out.device)
    nb = out[0].numel() * 4
    err = C.create_string_buffer(256)
    with torch.cuda.device(out.device):
        rc = L.pic_deposit_current_noalloc((C.c_int32 * 3)(nx, ny, nz), (C.c_double * 3)(*(float(v) for v in cell)),
                                           C.c_double(float(dt)), int(shape_order), C.c_int64(n), *args,
                                           *[C.c_void_p(out.data_ptr() + c * nb) for c in range(3)],
                                           C.c_void_p(st.cuda_stream), err, C.c_int64(len(err)))
    if rc != PIC_OK:
        raise PicError(rc, err.value.decode())
    return out
