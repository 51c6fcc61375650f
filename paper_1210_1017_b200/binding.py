"""Thin ctypes binding of libsph_b200.so - same names as include/sph_b200.h.

Argument marshalling only: every step of the path runs in the CUDA kernels.  PyTorch is used
for device memory (the workspace tensor), the stream and zero-copy views of the results.
There is NO fallback: importing this module without the built library raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsph_b200.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build the CUDA extension first "
        "(python -m paper_1210_1017_b200.build, or __graft_entry__.build()). "
        "There is no CPU fallback.")
_lib = C.CDLL(LIB_PATH)

SPH_MAX_SLABS = 16
SPH_OK = 0
(SPH_T_KEYS, SPH_T_SORT, SPH_T_GATHER, SPH_T_CELLS, SPH_T_HALO, SPH_T_MIGRATE, SPH_T_INTERACT,
 SPH_T_VERLET, SPH_T_DTREDUCE, SPH_T_COUNT) = range(10)
STAGE_NAMES = ["keys", "sort", "gather", "cells", "halo", "migrate", "interact", "verlet", "dt_reduce"]
SPH_OPT_INTERACT_VARIANT = 0
SPH_OPT_ADAPTIVE_DT = 1

EXPORTS = ["sph_workspace_bytes", "sph_init", "sph_set_state", "sph_set_slabs", "sph_slab_planes_from_x",
           "sph_sort_and_cells", "sph_build_halos", "sph_interact", "sph_interact_slab", "sph_step", "sph_time_step", "sph_step_adaptive", "sph_get_view",
           "sph_download", "sph_status", "sph_set_option", "sph_profile_enable", "sph_profile_read",
           "sph_pair_stats", "sph_launch_count", "sph_destroy", "sph_strerror", "sph_balance_slabs",
           "sph_download_resume", "sph_set_resume", "sph_last_cuda_error", "sph_fma_peak",
           "sph_cell_table_static", "sph_cell_table_static_error"]
SPH_ERR_STATIC_LIMIT = -8
SPH_STATIC_MAX_CELLS = 1 << 22
SPH_STATIC_SCRATCH_BYTES = 2098560


class sph_params(C.Structure):
    _fields_ = [("dp", C.c_float), ("h", C.c_float), ("rho0", C.c_float), ("c0", C.c_float),
                ("alpha", C.c_float), ("gamma", C.c_int), ("g", C.c_float * 3),
                ("mass_fluid", C.c_float), ("mass_bound", C.c_float),
                ("dom_min", C.c_float * 3), ("dom_max", C.c_float * 3),
                ("verlet_ns", C.c_int), ("kernel", C.c_int)]


class sph_particles(C.Structure):
    _fields_ = [("n", C.c_uint64), ("pos", C.c_void_p), ("vel", C.c_void_p), ("rho", C.c_void_p),
                ("type", C.c_void_p), ("prev_slab", C.c_void_p), ("on_device", C.c_int)]


class sph_view(C.Structure):
    _fields_ = [("n", C.c_uint64), ("nc", C.c_int32 * 3), ("ncells", C.c_uint32), ("cell_bits", C.c_int32),
                ("n_slabs", C.c_int32), ("step_index", C.c_uint64),
                ("pos4", C.c_void_p), ("velrho4", C.c_void_p), ("velrhoM1_4", C.c_void_p), ("acc4", C.c_void_p),
                ("idt", C.c_void_p), ("keyword", C.c_void_p), ("cell_begin", C.c_void_p),
                ("slab_begin", C.c_void_p), ("halo_offset", C.c_void_p), ("halo_pos4", C.c_void_p),
                ("halo_velrho4", C.c_void_p), ("halo_idt", C.c_void_p), ("mig_total", C.c_void_p),
                ("migrants", C.c_void_p), ("mig_count", C.c_void_p), ("mumax", C.c_void_p)]


_lib.sph_workspace_bytes.restype = C.c_size_t
_lib.sph_workspace_bytes.argtypes = [C.POINTER(sph_params), C.c_uint64, C.c_int]
_lib.sph_init.restype = C.c_int
_lib.sph_init.argtypes = [C.POINTER(C.c_void_p), C.POINTER(sph_params), C.POINTER(sph_particles), C.c_int,
                          C.c_void_p, C.c_size_t, C.c_void_p]
_lib.sph_set_state.restype = C.c_int
_lib.sph_set_state.argtypes = [C.c_void_p, C.POINTER(sph_particles)]
_lib.sph_set_slabs.restype = C.c_int
_lib.sph_set_slabs.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.c_int]
_lib.sph_slab_planes_from_x.restype = C.c_int
_lib.sph_slab_planes_from_x.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.c_int, C.POINTER(C.c_int32)]
for _name in ("sph_sort_and_cells", "sph_interact", "sph_status"):
    getattr(_lib, _name).restype = C.c_int
    getattr(_lib, _name).argtypes = [C.c_void_p]
_lib.sph_interact_slab.restype = C.c_int
_lib.sph_interact_slab.argtypes = [C.c_void_p, C.c_int]
_lib.sph_build_halos.restype = C.c_int
_lib.sph_build_halos.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.c_int]
_lib.sph_step.restype = C.c_int
_lib.sph_step.argtypes = [C.c_void_p, C.c_float]
_lib.sph_time_step.restype = C.c_int
_lib.sph_time_step.argtypes = [C.c_void_p, C.c_float, C.POINTER(C.c_float), C.POINTER(C.c_float),
                               C.POINTER(C.c_float)]
_lib.sph_step_adaptive.restype = C.c_int
_lib.sph_step_adaptive.argtypes = [C.c_void_p, C.c_float, C.POINTER(C.c_float)]
_lib.sph_get_view.restype = C.c_int
_lib.sph_get_view.argtypes = [C.c_void_p, C.POINTER(sph_view)]
_lib.sph_download.restype = C.c_int
_lib.sph_download.argtypes = [C.c_void_p] + [C.c_void_p] * 5
_lib.sph_set_option.restype = C.c_int
_lib.sph_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int]
_lib.sph_profile_enable.restype = C.c_int
_lib.sph_profile_enable.argtypes = [C.c_void_p, C.c_int]
_lib.sph_profile_read.restype = C.c_int
_lib.sph_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_float), C.POINTER(C.c_int)]
_lib.sph_pair_stats.restype = C.c_int
_lib.sph_pair_stats.argtypes = [C.c_void_p, C.POINTER(C.c_uint64)]
_lib.sph_launch_count.restype = C.c_int
_lib.sph_launch_count.argtypes = [C.c_void_p, C.POINTER(C.c_uint64)]
_lib.sph_balance_slabs.restype = C.c_int
_lib.sph_balance_slabs.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int32)]
_lib.sph_download_resume.restype = C.c_int
_lib.sph_download_resume.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_uint64)]
_lib.sph_set_resume.restype = C.c_int
_lib.sph_set_resume.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64, C.c_int]
_lib.sph_last_cuda_error.restype = C.c_char_p
_lib.sph_last_cuda_error.argtypes = [C.c_void_p]
_lib.sph_fma_peak.restype = C.c_int
_lib.sph_fma_peak.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_double)]
_lib.sph_cell_table_static.restype = C.c_int
_lib.sph_cell_table_static.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_void_p, C.c_void_p]
_lib.sph_cell_table_static_error.restype = C.c_char_p
_lib.sph_cell_table_static_error.argtypes = []
_lib.sph_destroy.restype = None
_lib.sph_destroy.argtypes = [C.c_void_p]
_lib.sph_strerror.restype = C.c_char_p
_lib.sph_strerror.argtypes = [C.c_int]


class SphError(RuntimeError):
    def __init__(self, code: int, detail: str = ""):
        self.code = code
        super().__init__(f"libsph_b200: {sph_strerror(code)} ({code})" + (f": {detail}" if detail else ""))


def sph_strerror(code: int) -> str:
    return _lib.sph_strerror(int(code)).decode()


def _check(rc: int) -> None:
    if rc != SPH_OK:
        raise SphError(rc)


def sph_cell_table_static(keyword, ncells: int, cell_begin, stream=None) -> None:
    """Cell table of a sorted keyword array for callers that cannot allocate device memory (they hold
    only borrowed pointers, or their process has no free GPU memory left to ask for): the scratch is a
    fixed array inside the library, so ncells is limited to SPH_STATIC_MAX_CELLS and calls on one GPU must
    not overlap.  keyword: int32 CUDA tensor of n sorted keywords (e.g. view_tensors()["keyword"]);
    cell_begin: int32 CUDA tensor of ncells + 1 entries on the same device, written in full.  The call is
    enqueued on ``stream`` (default: torch's current stream of that device).  See include/sph_b200.h."""
    import torch
    assert keyword.is_cuda and cell_begin.is_cuda and keyword.device == cell_begin.device
    assert keyword.dtype == torch.int32 and cell_begin.dtype == torch.int32
    assert keyword.is_contiguous() and cell_begin.is_contiguous()
    assert cell_begin.numel() == int(ncells) + 1
    with torch.cuda.device(keyword.device):
        st = stream if stream is not None else torch.cuda.current_stream(keyword.device)
        rc = _lib.sph_cell_table_static(C.c_void_p(keyword.data_ptr() if keyword.numel() else None),
                                        int(keyword.numel()), int(ncells), C.c_void_p(cell_begin.data_ptr()),
                                        C.c_void_p(st.cuda_stream))
    if rc != SPH_OK:
        raise SphError(rc, _lib.sph_cell_table_static_error().decode())


def make_params(P: dict) -> sph_params:
    p = sph_params()
    p.dp, p.h, p.rho0, p.c0, p.alpha = P["dp"], P["h"], P["rho0"], P["c0"], P["alpha"]
    p.gamma = int(P["gamma"])
    p.g[:] = P["g"]
    p.mass_fluid, p.mass_bound = P["mass_fluid"], P["mass_bound"]
    p.dom_min[:] = P["dom_min"]
    p.dom_max[:] = P["dom_max"]
    p.verlet_ns = int(P.get("verlet_ns", 40))
    p.kernel = int(P.get("kernel", 0))
    return p


def sph_workspace_bytes(params: sph_params, n_max: int, max_slabs: int) -> int:
    return int(_lib.sph_workspace_bytes(C.byref(params), int(n_max), int(max_slabs)))


def _ptr(a):
    """HOST numpy array or DEVICE torch tensor -> (address, on_device, keepalive)."""
    if a is None:
        return None, None, None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data, 0, a
    import torch
    assert isinstance(a, torch.Tensor) and a.is_contiguous()
    return a.data_ptr(), 1 if a.is_cuda else 0, a


def _particles(n, pos, vel, rho, typ, prev_slab):
    part = sph_particles()
    part.n = int(n)
    keep = []
    dev = None
    for name, arr, dt in (("pos", pos, "float32"), ("vel", vel, "float32"), ("rho", rho, "float32"),
                          ("type", typ, "uint8"), ("prev_slab", prev_slab, "uint8")):
        if arr is None:
            setattr(part, name, None)
            continue
        if isinstance(arr, np.ndarray):
            arr = np.ascontiguousarray(arr, dtype=dt)
        addr, on_dev, k = _ptr(arr)
        assert dev is None or dev == on_dev, "all particle arrays must live on the same side"
        dev = on_dev
        keep.append(k)
        setattr(part, name, addr)
    part.on_device = int(dev or 0)
    return part, keep


class Sph:
    """One context of the C library plus the torch-owned workspace and stream."""

    def __init__(self, P: dict, pos, vel, rho, typ=None, prev_slab=None, max_slabs: int = SPH_MAX_SLABS,
                 device: str = "cuda:0", stream=None):
        import torch
        self._ctx = C.c_void_p()
        if not torch.cuda.is_available():
            raise RuntimeError("libsph_b200 needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.params = make_params(P)
        self.n = int(rho.shape[0])
        nbytes = sph_workspace_bytes(self.params, self.n, max_slabs)
        if nbytes == 0:
            raise SphError(-3)
        torch.cuda.set_device(self.device)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        self._ws_off = (-self.workspace.data_ptr()) % 256
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._ctx = C.c_void_p()
        part, keep = _particles(self.n, pos, vel, rho, typ, prev_slab)
        _check(_lib.sph_init(C.byref(self._ctx), C.byref(self.params), C.byref(part), int(max_slabs),
                             C.c_void_p(self.workspace.data_ptr() + self._ws_off), nbytes,
                             C.c_void_p(self.stream.cuda_stream)))
        del keep

    # ---- the C ABI, same names -------------------------------------------------------------
    def sph_set_state(self, pos, vel, rho, typ=None, prev_slab=None):
        part, keep = _particles(self.n, pos, vel, rho, typ, prev_slab)
        _check(_lib.sph_set_state(self._ctx, C.byref(part)))

    def sph_set_slabs(self, planes):
        arr = (C.c_int32 * len(planes))(*[int(x) for x in planes])
        _check(_lib.sph_set_slabs(self._ctx, arr, len(planes) - 1))

    def sph_slab_planes_from_x(self, x_bounds):
        S = len(x_bounds) - 1
        xb = (C.c_float * (S + 1))(*[float(x) for x in x_bounds])
        out = (C.c_int32 * (S + 1))()
        _check(_lib.sph_slab_planes_from_x(self._ctx, xb, S, out))
        return list(out)

    def sph_sort_and_cells(self):
        _check(_lib.sph_sort_and_cells(self._ctx))

    def sph_build_halos(self, planes=None):
        if planes is None:
            _check(_lib.sph_build_halos(self._ctx, None, 0))
        else:
            arr = (C.c_int32 * len(planes))(*[int(x) for x in planes])
            _check(_lib.sph_build_halos(self._ctx, arr, len(planes) - 1))

    def sph_interact(self):
        _check(_lib.sph_interact(self._ctx))

    def sph_interact_slab(self, slab: int):
        _check(_lib.sph_interact_slab(self._ctx, int(slab)))

    def sph_step(self, dt: float):
        _check(_lib.sph_step(self._ctx, float(dt)))

    def sph_time_step(self, cfl: float):
        """(dt, amax_slab, smax_slab): variable time step and the per-sub-domain maxima it came from."""
        dt = C.c_float(0.0)
        am = (C.c_float * SPH_MAX_SLABS)()
        sm = (C.c_float * SPH_MAX_SLABS)()
        _check(_lib.sph_time_step(self._ctx, float(cfl), C.byref(dt), am, sm))
        S = int(self.sph_get_view().n_slabs)
        return float(dt.value), np.array(am[:S], dtype=np.float32), np.array(sm[:S], dtype=np.float32)

    def sph_step_adaptive(self, cfl: float) -> float:
        dt = C.c_float(0.0)
        _check(_lib.sph_step_adaptive(self._ctx, float(cfl), C.byref(dt)))
        return float(dt.value)

    def sph_status(self) -> int:
        return int(_lib.sph_status(self._ctx))

    def sph_set_option(self, option: int, value: int):
        _check(_lib.sph_set_option(self._ctx, int(option), int(value)))

    def sph_profile_enable(self, enable: bool):
        _check(_lib.sph_profile_enable(self._ctx, int(bool(enable))))

    def sph_profile_read(self):
        ms = (C.c_float * SPH_T_COUNT)()
        cnt = (C.c_int * SPH_T_COUNT)()
        _check(_lib.sph_profile_read(self._ctx, ms, cnt))
        return {STAGE_NAMES[k]: (float(ms[k]), int(cnt[k])) for k in range(SPH_T_COUNT)}

    def sph_pair_stats(self):
        """(candidate pairs examined by the 27-cell search, pairs with 0 < r < 2h)."""
        out = (C.c_uint64 * 2)()
        _check(_lib.sph_pair_stats(self._ctx, out))
        return int(out[0]), int(out[1])

    def sph_balance_slabs(self, n_slabs: int):
        """Planes (list of n_slabs + 1 cell-plane indices) that equalise the owned counts."""
        out = (C.c_int32 * (int(n_slabs) + 1))()
        _check(_lib.sph_balance_slabs(self._ctx, int(n_slabs), out))
        return [int(x) for x in out]

    def sph_download_resume(self):
        """(vel_m1 (n,3), rho_m1 (n,), step_index): the Verlet n-1 state in id order."""
        vel = np.empty((self.n, 3), dtype=np.float32)
        rho = np.empty(self.n, dtype=np.float32)
        k = C.c_uint64(0)
        _check(_lib.sph_download_resume(self._ctx, vel.ctypes.data, rho.ctypes.data, C.byref(k)))
        return vel, rho, int(k.value)

    def sph_set_resume(self, vel_m1, rho_m1, step_index: int):
        a, dev_a, k1 = _ptr(np.ascontiguousarray(vel_m1, dtype=np.float32) if isinstance(vel_m1, np.ndarray) else vel_m1)
        b, dev_b, k2 = _ptr(np.ascontiguousarray(rho_m1, dtype=np.float32) if isinstance(rho_m1, np.ndarray) else rho_m1)
        assert dev_a == dev_b
        _check(_lib.sph_set_resume(self._ctx, a, b, int(step_index), int(dev_a)))

    def sph_last_cuda_error(self) -> str:
        return _lib.sph_last_cuda_error(self._ctx).decode()

    def sph_fma_peak(self, variant: int = 0, iters: int = 4096) -> float:
        """Measured FP32 TFLOP/s of a register-resident FMA chain (0 = FFMA, 1 = packed FFMA2)."""
        out = C.c_double(0.0)
        _check(_lib.sph_fma_peak(self._ctx, int(variant), int(iters), C.byref(out)))
        return float(out.value)

    def sph_launch_count(self) -> int:
        out = C.c_uint64(0)
        _check(_lib.sph_launch_count(self._ctx, C.byref(out)))
        return int(out.value)

    def sph_get_view(self) -> sph_view:
        v = sph_view()
        _check(_lib.sph_get_view(self._ctx, C.byref(v)))
        return v

    def sph_download(self, pos=True, vel=True, rho=True, acc=True, drho=True, pinned=None):
        """HOST arrays in id order: dict of numpy arrays (or views of ``pinned`` torch buffers)."""
        n = self.n
        out, ptrs = {}, []
        for name, want, shape in (("pos", pos, (n, 3)), ("vel", vel, (n, 3)), ("rho", rho, (n,)),
                                  ("acc", acc, (n, 3)), ("drho", drho, (n,))):
            if not want:
                ptrs.append(None)
                continue
            if pinned is not None and name in pinned:
                a = pinned[name].numpy()
            else:
                a = np.empty(shape, dtype=np.float32)
            out[name] = a
            ptrs.append(a.ctypes.data)
        _check(_lib.sph_download(self._ctx, *ptrs))
        return out

    def sph_destroy(self):
        if getattr(self, "_ctx", None):
            _lib.sph_destroy(self._ctx)
            self._ctx = C.c_void_p()

    __del__ = sph_destroy

    # ---- zero-copy torch views of the borrowed device pointers ---------------------------------
    def _wrap(self, addr: int, count: int, dtype, cols: int = 0):
        torch = self.torch
        esz = torch.empty(0, dtype=dtype).element_size()
        off = addr - self.workspace.data_ptr()
        nbytes = count * esz * (cols if cols else 1)
        t = self.workspace[off:off + nbytes].view(dtype)
        return t.view(count, cols) if cols else t

    def view_tensors(self) -> dict:
        """Sorted-order device arrays as torch tensors aliasing the workspace (no copies)."""
        torch = self.torch
        v = self.sph_get_view()
        n, S = int(v.n), int(v.n_slabs)
        i32 = torch.int32
        d = dict(view=v,
                 pos4=self._wrap(v.pos4, n, torch.float32, 4),
                 velrho4=self._wrap(v.velrho4, n, torch.float32, 4),
                 velrhoM1_4=self._wrap(v.velrhoM1_4, n, torch.float32, 4),
                 acc4=self._wrap(v.acc4, n, torch.float32, 4),
                 idt=self._wrap(v.idt, n, i32), keyword=self._wrap(v.keyword, n, i32),
                 cell_begin=self._wrap(v.cell_begin, int(v.ncells) + 1, i32),
                 slab_begin=self._wrap(v.slab_begin, S + 1, i32),
                 halo_offset=self._wrap(v.halo_offset, 2 * S + 1, i32),
                 mig_total=self._wrap(v.mig_total, 1, i32),
                 mig_count=self._wrap(v.mig_count, 2 * S, i32).view(S, 2),
                 mumax=self._wrap(v.mumax, n, torch.float32))
        self.torch.cuda.current_stream(self.device).synchronize()
        self.stream.synchronize()
        nh = int(d["halo_offset"][-1].item()) if S > 1 else 0
        d["halo_pos4"] = self._wrap(v.halo_pos4, nh, torch.float32, 4)
        d["halo_velrho4"] = self._wrap(v.halo_velrho4, nh, torch.float32, 4)
        d["halo_idt"] = self._wrap(v.halo_idt, nh, i32)
        nm = int(d["mig_total"].item()) if S > 1 else 0
        d["migrants"] = self._wrap(v.migrants, nm, i32, 4)
        return d
