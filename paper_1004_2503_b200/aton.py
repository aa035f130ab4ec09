"""Thin ctypes binding of the C ABI in include/aton.h: argument marshalling only.

Every step of the path runs in libaton.so's CUDA kernels.  torch supplies device memory for the
caller-side tensors and the CUDA stream.  There is no CPU fallback: a missing library or a machine
without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libaton.so")

OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, -1, -2, -3, -4

EXPORTS = ("aton_init", "aton_set_fields", "aton_set_sources", "aton_courant_dt", "aton_step",
           "aton_get_fields", "aton_reduce", "aton_set_kernel", "aton_launch_count", "aton_set_timing",
           "aton_kernel_time", "aton_fixup_time", "aton_init_slab", "aton_halo_pack", "aton_halo_unpack", "aton_set_mean_density",
           "aton_reduce_sums", "aton_diag_from_sums", "aton_set_mean_from_sums", "aton_comm_unique_id", "aton_comm_init",
           "aton_step_slab", "aton_reduce_global", "aton_sync_mean_density", "aton_clumping_blocks", "aton_histogram2d",
           "aton_set_star_sources", "aton_thomson_tau", "aton_field_sums_noalloc", "aton_free", "aton_last_error")
Q_NH, Q_X, Q_NEUTRAL, Q_T, Q_N, Q_GAMMA = range(6)
COMM_ID_BYTES = 128
NSUMS = 15
NOALLOC_NSUMS = 12


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int)]


class Box(C.Structure):
    _fields_ = [("lx_cm", C.c_double)]


class Params(C.Structure):
    _fields_ = [("c_cm_s", C.c_double), ("sigma_n", C.c_double), ("sigma_e", C.c_double),
                ("e_photon_eV", C.c_double), ("recomb_case", C.c_int), ("cooling", C.c_int),
                ("coll_ion", C.c_int), ("clump_model", C.c_int), ("clump_a", C.c_double),
                ("clump_b", C.c_double), ("redshift", C.c_double), ("eps_sub", C.c_double),
                ("max_sub", C.c_int), ("clump_i_a", C.c_double), ("clump_i_b", C.c_double), ("flux", C.c_int)]


class Diag(C.Structure):
    _fields_ = [("x_vol", C.c_double), ("x_mass", C.c_double), ("gamma_vol", C.c_double),
                ("gamma_mass", C.c_double), ("photons_total", C.c_double), ("T_vol", C.c_double),
                ("f_max", C.c_double), ("N_min", C.c_double), ("frac_x_half", C.c_double),
                ("n_nonfinite", C.c_longlong), ("subcycles_total", C.c_longlong),
                ("subcycles_max", C.c_longlong), ("cells_subcycled", C.c_longlong),
                ("steps_done", C.c_longlong), ("time_s", C.c_double), ("cells_fp64", C.c_longlong)]


class AtonError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"aton error {code}: {msg}")
        self.code = code


_lib = None


def load_library(path: Optional[str] = None):
    """dlopen libaton.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} not found: build it with `python -m paper_1004_2503_b200.build` "
                                "(there is no CPU fallback)")
    L = C.CDLL(path)
    vp, fp, dp = C.c_void_p, C.c_void_p, C.c_void_p
    L.aton_init.restype = C.c_int
    L.aton_init.argtypes = [C.POINTER(vp), C.POINTER(Grid), C.POINTER(Box), C.POINTER(Params), vp]
    L.aton_set_fields.restype = C.c_int
    L.aton_set_fields.argtypes = [vp] + [fp] * 7 + [C.c_int]
    L.aton_set_sources.restype = C.c_int
    L.aton_set_sources.argtypes = [vp, C.c_longlong, fp, dp, C.c_int]
    L.aton_courant_dt.restype = C.c_double
    L.aton_courant_dt.argtypes = [vp, C.c_double]
    L.aton_step.restype = C.c_int
    L.aton_step.argtypes = [vp, C.c_double, C.c_int]
    L.aton_get_fields.restype = C.c_int
    L.aton_get_fields.argtypes = [vp] + [fp] * 7 + [C.c_int]
    L.aton_reduce.restype = C.c_int
    L.aton_reduce.argtypes = [vp, C.POINTER(Diag)]
    L.aton_set_kernel.restype = C.c_int
    L.aton_set_kernel.argtypes = [vp, C.c_int, C.c_int, C.c_int]
    L.aton_launch_count.restype = C.c_longlong
    L.aton_launch_count.argtypes = [vp]
    L.aton_set_timing.restype = C.c_int
    L.aton_set_timing.argtypes = [vp, C.c_int]
    L.aton_kernel_time.restype = C.c_int
    L.aton_kernel_time.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    L.aton_fixup_time.restype = C.c_int
    L.aton_fixup_time.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    L.aton_init_slab.restype = C.c_int
    L.aton_init_slab.argtypes = [C.POINTER(vp), C.POINTER(Grid), C.POINTER(Box), C.POINTER(Params), vp, C.c_int, C.c_int]
    L.aton_halo_pack.restype = C.c_int
    L.aton_halo_pack.argtypes = [vp, fp, fp]
    L.aton_halo_unpack.restype = C.c_int
    L.aton_halo_unpack.argtypes = [vp, fp, fp]
    L.aton_set_mean_density.restype = C.c_int
    L.aton_set_mean_density.argtypes = [vp, C.c_double]
    L.aton_reduce_sums.restype = C.c_int
    L.aton_reduce_sums.argtypes = [vp, C.POINTER(C.c_double), C.c_int]
    L.aton_diag_from_sums.restype = C.c_int
    L.aton_diag_from_sums.argtypes = [vp, C.POINTER(C.c_double), C.c_int, C.POINTER(Diag)]
    L.aton_set_mean_from_sums.restype = C.c_int
    L.aton_set_mean_from_sums.argtypes = [vp, C.POINTER(C.c_double), C.c_int]
    L.aton_comm_unique_id.restype = C.c_int
    L.aton_comm_unique_id.argtypes = [C.c_char_p, C.c_int]
    L.aton_comm_init.restype = C.c_int
    L.aton_comm_init.argtypes = [vp, C.c_char_p, C.c_int, C.c_int, C.c_int]
    L.aton_step_slab.restype = C.c_int
    L.aton_step_slab.argtypes = [vp, C.c_double, C.c_int]
    L.aton_reduce_global.restype = C.c_int
    L.aton_reduce_global.argtypes = [vp, C.POINTER(Diag)]
    L.aton_sync_mean_density.restype = C.c_int
    L.aton_sync_mean_density.argtypes = [vp]
    L.aton_clumping_blocks.restype = C.c_int
    L.aton_clumping_blocks.argtypes = [vp, C.c_int, fp, fp, fp, fp, C.c_int]
    L.aton_histogram2d.restype = C.c_int
    L.aton_histogram2d.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int] + [C.c_double] * 4 + [C.c_int, C.c_int, vp, vp, C.c_int]
    L.aton_set_star_sources.restype = C.c_int
    L.aton_set_star_sources.argtypes = [vp, C.c_longlong, fp, dp, dp, dp] + [C.c_double] * 6 + [C.c_int]
    L.aton_thomson_tau.restype = C.c_int
    L.aton_thomson_tau.argtypes = [vp, C.c_longlong, dp, dp, C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double)]
    L.aton_field_sums_noalloc.restype = C.c_int
    L.aton_field_sums_noalloc.argtypes = [fp, fp, fp, fp, fp, fp, fp, C.c_longlong, C.c_double, vp, dp]
    L.aton_free.restype = None
    L.aton_free.argtypes = [vp]
    L.aton_last_error.restype = C.c_char_p
    L.aton_last_error.argtypes = [vp]
    _lib = L
    return L


def make_params(d: Dict[str, float]) -> Params:
    p = Params()
    for k, _ in Params._fields_:
        if k in d:
            setattr(p, k, type(getattr(p, k))(d[k]))
    return p


def _ptr(t: Optional[torch.Tensor], n: int, dtype, want_cuda: bool):
    if t is None:
        return None
    if t.dtype != dtype or not t.is_contiguous() or t.numel() != n:
        raise ValueError(f"expected a contiguous {dtype} tensor of {n} elements")
    if t.is_cuda != want_cuda:
        raise ValueError("all tensors of one call must live on the same side (host or device)")
    return C.c_void_p(t.data_ptr())


class Aton:
    """One simulation context (aton_t).  Methods mirror the C entry points one to one."""

    def __init__(self, nx: int, ny: int, nz: int, lx_cm: float, params: Dict[str, float],
                 stream: Optional[torch.cuda.Stream] = None, slab=None):
        """`slab` = (z_begin, nz_local): aton_init_slab on planes [z_begin, z_begin + nz_local) of the global grid."""
        self._L = load_library()
        self._h = C.c_void_p()
        nz_own = nz if slab is None else int(slab[1])
        self.shape = (nz_own, ny, nx)
        self.ncell = nx * ny * nz_own
        self.plane = nx * ny
        self._stream = stream
        sp = C.c_void_p(stream.cuda_stream if stream is not None
                        else (torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0))
        g, b, p = Grid(nx, ny, nz), Box(lx_cm), make_params(params)
        if slab is None:
            rc = self._L.aton_init(C.byref(self._h), C.byref(g), C.byref(b), C.byref(p), sp)
        else:
            rc = self._L.aton_init_slab(C.byref(self._h), C.byref(g), C.byref(b), C.byref(p), sp, int(slab[0]), int(slab[1]))
        if rc != OK:
            self._h = C.c_void_p()
            raise AtonError(rc, self._L.aton_last_error(None).decode())

    # -- plumbing
    def _check(self, rc: int):
        if rc != OK:
            raise AtonError(rc, self._L.aton_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.aton_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C entry points
    def set_fields(self, nH, x, T, N=None, Fx=None, Fy=None, Fz=None):
        dev = nH.is_cuda
        ptrs = [_ptr(t, self.ncell, torch.float32, dev) for t in (nH, x, T, N, Fx, Fy, Fz)]
        self._check(self._L.aton_set_fields(self._h, *ptrs, int(dev)))

    def set_sources(self, pos: Optional[torch.Tensor], rate: Optional[torch.Tensor]):
        n = 0 if rate is None else rate.numel()
        if n == 0:
            self._check(self._L.aton_set_sources(self._h, 0, None, None, 0))
            return
        dev = pos.is_cuda
        self._check(self._L.aton_set_sources(self._h, n, _ptr(pos, 3 * n, torch.float32, dev),
                                             _ptr(rate, n, torch.float64, dev), int(dev)))

    def courant_dt(self, courant: float = 0.8) -> float:
        return float(self._L.aton_courant_dt(self._h, courant))

    def step(self, dt: float, n_steps: int = 1):
        self._check(self._L.aton_step(self._h, float(dt), int(n_steps)))

    def get_fields(self, device=None, names=("nH", "x", "T", "N", "Fx", "Fy", "Fz"), out=None) -> Dict[str, torch.Tensor]:
        """Download the named fields into new tensors (on `device`, default cuda) or into `out`."""
        order = ("nH", "x", "T", "N", "Fx", "Fy", "Fz")
        if out is None:
            device = torch.device(device or "cuda")
            out = {k: torch.empty(self.shape, dtype=torch.float32, device=device,
                                  pin_memory=(device.type == "cpu")) for k in names}
        dev = next(iter(out.values())).is_cuda
        ptrs = [_ptr(out.get(k), self.ncell, torch.float32, dev) if k in out else None for k in order]
        self._check(self._L.aton_get_fields(self._h, *ptrs, int(dev)))
        return out

    def reduce(self) -> Dict[str, float]:
        d = Diag()
        self._check(self._L.aton_reduce(self._h, C.byref(d)))
        return {k: getattr(d, k) for k, _ in Diag._fields_}

    def set_kernel(self, variant: int, tile_y: int = 0, tile_z: int = 0):
        self._check(self._L.aton_set_kernel(self._h, variant, tile_y, tile_z))

    def halo_pack(self, send_lo: torch.Tensor, send_hi: torch.Tensor):
        self._check(self._L.aton_halo_pack(self._h, _ptr(send_lo, 4 * self.plane, torch.float32, True),
                                           _ptr(send_hi, 4 * self.plane, torch.float32, True)))

    def halo_unpack(self, recv_lo: torch.Tensor, recv_hi: torch.Tensor):
        self._check(self._L.aton_halo_unpack(self._h, _ptr(recv_lo, 4 * self.plane, torch.float32, True),
                                             _ptr(recv_hi, 4 * self.plane, torch.float32, True)))

    def set_mean_density(self, nH_mean: float):
        self._check(self._L.aton_set_mean_density(self._h, float(nH_mean)))

    def reduce_sums(self):
        buf = (C.c_double * NSUMS)()
        self._check(self._L.aton_reduce_sums(self._h, buf, NSUMS))
        return list(buf)

    def diag_from_sums(self, sums) -> Dict[str, float]:
        """aton_diag_t formed by the library from raw sums the caller combined across slabs."""
        buf = (C.c_double * NSUMS)(*sums)
        d = Diag()
        self._check(self._L.aton_diag_from_sums(self._h, buf, NSUMS, C.byref(d)))
        return {k: getattr(d, k) for k, _ in Diag._fields_}

    def set_mean_from_sums(self, sums):
        buf = (C.c_double * NSUMS)(*sums)
        self._check(self._L.aton_set_mean_from_sums(self._h, buf, NSUMS))

    def comm_init(self, comm_id: Optional[bytes], rank: int, world: int):
        """aton_comm_init: `comm_id` = the bytes of comm_unique_id() from rank 0 (None only for world == 1)."""
        self._check(self._L.aton_comm_init(self._h, comm_id, COMM_ID_BYTES if comm_id is not None else 0, rank, world))

    def step_slab(self, dt: float, n_steps: int = 1):
        self._check(self._L.aton_step_slab(self._h, float(dt), int(n_steps)))

    def reduce_global(self) -> Dict[str, float]:
        d = Diag()
        self._check(self._L.aton_reduce_global(self._h, C.byref(d)))
        return {k: getattr(d, k) for k, _ in Diag._fields_}

    def sync_mean_density(self):
        self._check(self._L.aton_sync_mean_density(self._h))

    def clumping_blocks(self, block: int = 8, device="cuda") -> Dict[str, torch.Tensor]:
        """aton_clumping_blocks: dict of [nz/b, ny/b, nx/b] float32 tensors nH, x, C_R, C_I."""
        nz, ny, nx = self.shape
        shape = (nz // block, ny // block, nx // block)
        dev = torch.device(device)
        out = {k: torch.empty(shape, dtype=torch.float32, device=dev) for k in ("nH", "x", "C_R", "C_I")}
        n = shape[0] * shape[1] * shape[2]
        self._check(self._L.aton_clumping_blocks(self._h, int(block), *[_ptr(out[k], n, torch.float32, dev.type == "cuda")
                                                                          for k in ("nH", "x", "C_R", "C_I")], int(dev.type == "cuda")))
        return out

    def histogram2d(self, qa: int, qb: int, log_a: bool, log_b: bool, a_range, b_range, na: int, nb: int):
        """aton_histogram2d: (counts[nb, na] int64 CPU tensor, number of cells outside the ranges)."""
        counts = torch.zeros((nb, na), dtype=torch.int64)
        outside = C.c_longlong(0)
        self._check(self._L.aton_histogram2d(self._h, qa, qb, int(log_a), int(log_b), float(a_range[0]), float(a_range[1]),
                                             float(b_range[0]), float(b_range[1]), na, nb, C.c_void_p(counts.data_ptr()),
                                             C.cast(C.byref(outside), C.c_void_p), 0))
        return counts, int(outside.value)

    def set_star_sources(self, pos, age, lifetime, nbaryons, photons_per_baryon, t_p, t_p1, f_esc, a_b, k_b):
        n = age.numel()
        dev = pos.is_cuda
        self._check(self._L.aton_set_star_sources(self._h, n, _ptr(pos, 3 * n, torch.float32, dev),
                                                  *[_ptr(t, n, torch.float64, dev) for t in (age, lifetime, nbaryons)],
                                                  float(photons_per_baryon), float(t_p), float(t_p1), float(f_esc), float(a_b),
                                                  float(k_b), int(dev)))

    def thomson_tau(self, z: torch.Tensor, x: torch.Tensor, nH0: float, H0: float, Om: float) -> float:
        n = z.numel()
        tau = C.c_double()
        self._check(self._L.aton_thomson_tau(self._h, n, _ptr(z, n, torch.float64, False), _ptr(x, n, torch.float64, False),
                                             float(nH0), float(H0), float(Om), C.byref(tau)))
        return tau.value

    def set_timing(self, on: bool):
        self._check(self._L.aton_set_timing(self._h, int(bool(on))))

    def kernel_time(self):
        """(sum of ms, launches) of the event-bracketed dominant step kernel since set_timing(True)."""
        ms, n = C.c_double(), C.c_longlong()
        self._check(self._L.aton_kernel_time(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def fixup_time(self):
        """(ms of step_fixup_kernel, ms of step_stiff_kernel, launches) summed since set_timing(True)."""
        ms, ms2, n = C.c_double(), C.c_double(), C.c_longlong()
        self._check(self._L.aton_fixup_time(self._h, C.byref(ms), C.byref(ms2), C.byref(n)))
        return ms.value, ms2.value, n.value

    def launch_count(self) -> int:
        return int(self._L.aton_launch_count(self._h))


def field_sums_noalloc(nH, x, T, N, Fx, Fy, Fz, out, c_cm_s: float = 0.0, stream=None):
    """aton_field_sums_noalloc: the raw sums of aton_reduce_sums of seven float32 CUDA tensors of equal size, written into
    `out` (a float64 CUDA tensor of NOALLOC_NSUMS elements) when the stream reaches the call.  Allocates nothing and does
    not synchronise; every call on a device shares one static scratch array (calls that overlap on the GPU race)."""
    L = load_library()
    n = nH.numel()
    for t in (nH, x, T, N, Fx, Fy, Fz):
        if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.numel() == n):
            raise ValueError("field_sums_noalloc: contiguous float32 CUDA tensors of one size, please")
    if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= NOALLOC_NSUMS):
        raise ValueError(f"field_sums_noalloc: `out` must be a float64 CUDA tensor of {NOALLOC_NSUMS} elements")
    st = (stream or torch.cuda.current_stream()).cuda_stream
    rc = L.aton_field_sums_noalloc(*[C.c_void_p(t.data_ptr()) for t in (nH, x, T, N, Fx, Fy, Fz)], n, float(c_cm_s),
                                   C.c_void_p(st), C.c_void_p(out.data_ptr()))
    if rc != OK:
        raise AtonError(rc, L.aton_last_error(None).decode())
    return out


def comm_unique_id() -> bytes:
    """An ncclUniqueId for aton_comm_init, as bytes (rank 0 calls this and distributes the result)."""
    buf = C.create_string_buffer(COMM_ID_BYTES)
    rc = load_library().aton_comm_unique_id(buf, COMM_ID_BYTES)
    if rc != OK:
        raise AtonError(rc, load_library().aton_last_error(None).decode())
    return buf.raw


def from_workload(w, stream=None, device="cuda") -> Aton:
    """Context initialised from a workloads.Workload (fields uploaded, sources set)."""
    a = Aton(w.n, w.n, w.n, w.box_cm, w.params, stream)
    f = [t.to(device).contiguous() for t in w.fields()]
    a.set_fields(*f)
    a.set_sources(w.src_pos.contiguous(), w.src_rate.contiguous())
    return a
