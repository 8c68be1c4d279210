"""Thin ctypes binding over libchemora.so (include/chemora.h): argument marshalling only -- every step of
the path runs in the library's CUDA kernels.  PyTorch is used for device memory (the library's allocator
callbacks hand out torch-owned buffers) and for the CUDA stream; nothing here computes.

There is no CPU fallback: `load()` raises if the library is missing and `Chemora(...)` raises
ChemoraError(CHEMORA_ECUDA) when no CUDA device is present.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libchemora.so")

SYS_WAVE, SYS_BSSN, SYS_WAVE1 = 0, 1, 2
BUF_U, BUF_YA, BUF_YB, BUF_S = 0, 1, 2, 3
BC_PERIODIC, BC_RADIATIVE = 0, 1
NUM_TILES = 9
OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, -1, -2, -3, -4

# every symbol include/chemora.h declares (tests check that the library exports all of them)
SYMBOLS = ["chemora_create", "chemora_set_param", "chemora_get_param", "chemora_layout", "chemora_state_ptr",
           "chemora_set_state", "chemora_get_state", "chemora_set_state_async", "chemora_get_state_async",
           "chemora_synchronize", "chemora_set_state_dev", "chemora_get_state_dev",
           "chemora_fill_ghosts", "chemora_rhs", "chemora_rk4_step", "chemora_rk3_step", "chemora_link_z",
           "chemora_rk4_step_group", "chemora_rk3_step_group", "chemora_set_boundary", "chemora_get_boundary", "chemora_radiative_rhs",
           "chemora_set_state_ghosted", "chemora_get_state_ghosted", "chemora_enforce_constraints", "chemora_energy", "chemora_set_variant",
           "chemora_get_variant", "chemora_variant_available", "chemora_selfcheck", "chemora_describe_device_error", "chemora_tile_shape", "chemora_tile_cost", "chemora_autotune", "chemora_launch_count",
           "chemora_kernel_info", "chemora_measure_box_fill", "chemora_timing", "chemora_timing_read", "chemora_measure_fp64_peak", "chemora_last_error", "chemora_destroy"]

_ALLOC_T = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)
_DEALLOC_T = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)

_lib = None


class ChemoraError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__("chemora error %d %s" % (code, msg))
        self.code = code


def load():
    """Load libchemora.so (built in-tree by paper_1307_6488_b200.build).  Fails loudly when missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ChemoraError(ESTATE, "libchemora.so not built: run `python -m paper_1307_6488_b200.build` "
                                   "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i, d, l = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_long
    ip, lp, dp = ctypes.POINTER(i), ctypes.POINTER(l), ctypes.POINTER(d)
    sig = {
        "chemora_create": [ctypes.POINTER(vp), i, i, i, i, i, i, d, vp, _ALLOC_T, _DEALLOC_T, vp],
        "chemora_set_param": [vp, ctypes.c_char_p, d],
        "chemora_get_param": [vp, ctypes.c_char_p, dp],
        "chemora_layout": [vp, ip, lp, lp, lp, lp, lp],
        "chemora_state_ptr": [vp, i, ctypes.POINTER(vp)],
        "chemora_set_state": [vp, vp], "chemora_get_state": [vp, vp],
        "chemora_set_state_dev": [vp, vp], "chemora_get_state_dev": [vp, vp],
        "chemora_fill_ghosts": [vp, vp], "chemora_rhs": [vp, vp, vp],
        "chemora_rk4_step": [vp, d],
        "chemora_rk3_step": [vp, d],
        "chemora_set_state_async": [vp, vp], "chemora_get_state_async": [vp, vp], "chemora_synchronize": [vp],
        "chemora_link_z": [vp, vp, vp],
        "chemora_set_boundary": [vp, i], "chemora_get_boundary": [vp, ip], "chemora_radiative_rhs": [vp, vp, vp],
        "chemora_set_state_ghosted": [vp, vp], "chemora_get_state_ghosted": [vp, vp],
        "chemora_rk4_step_group": [ctypes.POINTER(vp), i, d], "chemora_rk3_step_group": [ctypes.POINTER(vp), i, d],
        "chemora_tile_cost": [i, i, i, dp, lp, lp],
        "chemora_enforce_constraints": [vp, vp],
        "chemora_energy": [vp, vp, vp, dp],
        "chemora_set_variant": [vp, i, i], "chemora_get_variant": [vp, ip, ip],
        "chemora_tile_shape": [i, i, i, ip, ip, ip],
        "chemora_variant_available": [i, i, i, i],
        "chemora_selfcheck": [ctypes.c_char_p, ctypes.c_size_t],
        "chemora_describe_device_error": [ctypes.c_uint, ctypes.c_char_p, ctypes.c_size_t],
        "chemora_autotune": [vp, ip, ip, ctypes.POINTER(ctypes.c_float)],
        "chemora_launch_count": [vp],
        "chemora_kernel_info": [vp, ip, ip, ip],
        "chemora_measure_fp64_peak": [vp, dp],
        "chemora_measure_box_fill": [vp, i, ctypes.POINTER(ctypes.c_float)],
        "chemora_timing": [vp, i], "chemora_timing_read": [vp, dp, lp, dp, lp],
        "chemora_last_error": [vp], "chemora_destroy": [vp],
    }
    for name, args in sig.items():
        f = getattr(lib, name)
        f.argtypes = args
        f.restype = i
    lib.chemora_launch_count.restype = l
    lib.chemora_last_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def tile_shape(tile_id, system_id=SYS_BSSN, fused=1):
    a, b, c = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    rc = load().chemora_tile_shape(system_id, fused, tile_id, a, b, c)
    if rc:
        raise ChemoraError(rc)
    return a.value, b.value, c.value


def variant_available(system_id, fd_order, fused, tile_id):
    return bool(load().chemora_variant_available(system_id, fd_order, fused, tile_id))


def variants(system_id, fd_order, fused=1):
    """the tile ids that exist for a system, order and variant axis"""
    return [t for t in range(NUM_TILES) if variant_available(system_id, fd_order, fused, t)]


def selfcheck():
    """(number of launch plans checked, report line); raises if the validator rejects one.  Host only."""
    buf = ctypes.create_string_buffer(512)
    rc = load().chemora_selfcheck(buf, len(buf))
    if rc <= 0:
        raise ChemoraError(rc, buf.value.decode())
    return rc, buf.value.decode()


def describe_device_error(code):
    buf = ctypes.create_string_buffer(256)
    rc = load().chemora_describe_device_error(code, buf, len(buf))
    if rc:
        raise ChemoraError(rc)
    return buf.value.decode()


def step_group(blocks, dt, rk3=False):
    """one RK4 (or RK3) step of a group of z-linked blocks: chemora_rk4_step_group / chemora_rk3_step_group"""
    arr = (ctypes.c_void_p * len(blocks))(*[b._h for b in blocks])
    fn = blocks[0].lib.chemora_rk3_step_group if rk3 else blocks[0].lib.chemora_rk4_step_group
    blocks[0]._ck(fn(arr, len(blocks), float(dt)))


def tile_cost(fd_order, ghost, tile_id):
    """(sigma, requests, points) of the paper's tile cost model for a fused BSSN tile id; host arithmetic only"""
    s, r, n = ctypes.c_double(), ctypes.c_long(), ctypes.c_long()
    rc = load().chemora_tile_cost(fd_order, ghost, tile_id, ctypes.byref(s), ctypes.byref(r), ctypes.byref(n))
    if rc:
        raise ChemoraError(rc)
    return s.value, r.value, n.value


class Chemora:
    """One handle = one grid block on one GPU.  Methods mirror the C entry points one to one."""

    def __init__(self, nx, ny, nz, ghost, fd_order, system_id, dx, device="cuda:0", use_torch_alloc=True):
        import torch
        self._torch = torch
        self.lib = load()
        self._h = ctypes.c_void_p()
        self._owned = {}
        self.dims = (nx, ny, nz)
        self.ghost = ghost
        stream = 0
        if torch.cuda.is_available():
            self.device = torch.device(device)
            torch.cuda.set_device(self.device)
            stream = torch.cuda.current_stream(self.device).cuda_stream
        else:
            self.device = None

        def _alloc(nbytes, _ctx):
            try:
                t = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
            except Exception:
                return None
            self._owned[t.data_ptr()] = t
            return t.data_ptr()

        def _dealloc(ptr, _ctx):
            self._owned.pop(ptr, None)

        self._alloc_cb = _ALLOC_T(_alloc) if (use_torch_alloc and self.device is not None) else _ALLOC_T()
        self._dealloc_cb = _DEALLOC_T(_dealloc) if (use_torch_alloc and self.device is not None) else _DEALLOC_T()
        rc = self.lib.chemora_create(ctypes.byref(self._h), nx, ny, nz, ghost, fd_order, system_id, float(dx),
                                     ctypes.c_void_p(stream), self._alloc_cb, self._dealloc_cb, None)
        if rc:
            self._h = ctypes.c_void_p()
            raise ChemoraError(rc, "chemora_create failed")
        nv, pitch, ty, tz, vs, io = (ctypes.c_int(), ctypes.c_long(), ctypes.c_long(), ctypes.c_long(),
                                     ctypes.c_long(), ctypes.c_long())
        self._ck(self.lib.chemora_layout(self._h, nv, pitch, ty, tz, vs, io))
        self.nvars, self.pitch, self.tot_y, self.tot_z = nv.value, pitch.value, ty.value, tz.value
        self.var_stride, self.interior_offset = vs.value, io.value
        self.xoff = self.interior_offset % self.pitch      # x index of interior point 0 inside a row

    # -- helpers -------------------------------------------------------------------------------------
    def _ck(self, rc):
        if rc:
            raise ChemoraError(rc, (self.lib.chemora_last_error(self._h) or b"").decode())

    @staticmethod
    def _ptr(t):
        return ctypes.c_void_p(t if isinstance(t, int) else t.data_ptr())

    def new_state(self):
        """A zeroed device tensor in the padded layout [V, tot_z, tot_y, pitch] (torch owns it)."""
        return self._torch.zeros((self.nvars, self.tot_z, self.tot_y, self.pitch), dtype=self._torch.float64,
                                 device=self.device)

    def state_view(self, which=BUF_U):
        """One of the library's four buffers as a torch tensor [V, tot_z, tot_y, pitch] sharing its memory
        (possible because the buffers come from the torch allocator callbacks)."""
        p = self.state_ptr(which)
        if p not in self._owned:
            raise ChemoraError(ESTATE, "state_view needs use_torch_alloc=True")
        n = self.nvars * self.var_stride
        return self._owned[p].view(self._torch.float64)[:n].view(self.nvars, self.tot_z, self.tot_y, self.pitch)

    def state_ptr(self, which=BUF_U):
        p = ctypes.c_void_p()
        self._ck(self.lib.chemora_state_ptr(self._h, which, ctypes.byref(p)))
        return p.value

    def interior(self, padded):
        g, xo, (nx, ny, nz) = self.ghost, self.xoff, self.dims
        return padded[:, g:g + nz, g:g + ny, xo:xo + nx]

    def ghosted(self, padded):
        """the [V, nz+2g, ny+2g, nx+2g] part of a padded state (interior + ghosts, no row padding)"""
        g, xo, nx = self.ghost, self.xoff, self.dims[0]
        return padded[..., xo - g:xo + nx + g]

    # -- the C entry points ---------------------------------------------------------------------------
    def set_param(self, name, value):
        self._ck(self.lib.chemora_set_param(self._h, name.encode(), float(value)))

    def get_param(self, name):
        v = ctypes.c_double()
        self._ck(self.lib.chemora_get_param(self._h, name.encode(), v))
        return v.value

    def set_state(self, host_packed):
        a = np.ascontiguousarray(host_packed, dtype=np.float64)
        assert a.size == self.nvars * self.dims[0] * self.dims[1] * self.dims[2]
        self._ck(self.lib.chemora_set_state(self._h, ctypes.c_void_p(a.ctypes.data)))

    def get_state(self, out=None):
        nx, ny, nz = self.dims
        if out is None:
            out = np.empty((self.nvars, nz, ny, nx), dtype=np.float64)
        self._ck(self.lib.chemora_get_state(self._h, ctypes.c_void_p(out.ctypes.data)))
        return out

    def _host_ptr(self, a):
        """host pointer of a numpy array or a (pinned) CPU torch tensor, kept alive until synchronize()"""
        if not hasattr(self, "_inflight"):
            self._inflight = []
        self._inflight.append(a)
        if isinstance(a, np.ndarray):
            assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
            n, p = a.size, a.ctypes.data
        else:
            assert a.dtype == self._torch.float64 and a.is_contiguous() and not a.is_cuda
            n, p = a.numel(), a.data_ptr()
        assert n == self.nvars * self.dims[0] * self.dims[1] * self.dims[2]
        return ctypes.c_void_p(p)

    def set_state_async(self, host_packed):
        """queue the copy of a packed host state (page-locked for a real overlap) into U; see chemora.h"""
        self._ck(self.lib.chemora_set_state_async(self._h, self._host_ptr(host_packed)))

    def get_state_async(self, out):
        self._ck(self.lib.chemora_get_state_async(self._h, self._host_ptr(out)))

    def synchronize(self):
        self._ck(self.lib.chemora_synchronize(self._h))
        self._inflight = []

    def synchronize_quietly(self):
        """chemora_synchronize, return code instead of an exception (clears a pending device error word)"""
        return self.lib.chemora_synchronize(self._h)

    def set_state_dev(self, dev_packed):
        self._ck(self.lib.chemora_set_state_dev(self._h, self._ptr(dev_packed)))

    def get_state_dev(self, dev_packed):
        self._ck(self.lib.chemora_get_state_dev(self._h, self._ptr(dev_packed)))

    def fill_ghosts(self, dev_state):
        self._ck(self.lib.chemora_fill_ghosts(self._h, self._ptr(dev_state)))

    def rhs(self, dev_state, dev_rhs):
        self._ck(self.lib.chemora_rhs(self._h, self._ptr(dev_state), self._ptr(dev_rhs)))

    def rk4_step(self, dt):
        self._ck(self.lib.chemora_rk4_step(self._h, float(dt)))

    def rk3_step(self, dt):
        self._ck(self.lib.chemora_rk3_step(self._h, float(dt)))

    def link_z(self, lower=None, upper=None):
        """multi-block interface: the ghost z-planes come from the neighbour blocks' interiors (None: own images)"""
        self._ck(self.lib.chemora_link_z(self._h, lower._h if lower is not None else None,
                                         upper._h if upper is not None else None))

    def set_boundary(self, kind):
        self._ck(self.lib.chemora_set_boundary(self._h, int(kind)))

    def get_boundary(self):
        k = ctypes.c_int()
        self._ck(self.lib.chemora_get_boundary(self._h, ctypes.byref(k)))
        return k.value

    def radiative_rhs(self, dev_state, dev_rhs):
        self._ck(self.lib.chemora_radiative_rhs(self._h, self._ptr(dev_state), self._ptr(dev_rhs)))

    def set_state_ghosted(self, host_ghosted):
        g, (nx, ny, nz) = self.ghost, self.dims
        a = np.ascontiguousarray(host_ghosted, dtype=np.float64)
        assert a.shape == (self.nvars, nz + 2 * g, ny + 2 * g, nx + 2 * g)
        self._ck(self.lib.chemora_set_state_ghosted(self._h, a.ctypes.data_as(ctypes.c_void_p)))

    def get_state_ghosted(self):
        g, (nx, ny, nz) = self.ghost, self.dims
        out = np.empty((self.nvars, nz + 2 * g, ny + 2 * g, nx + 2 * g), dtype=np.float64)
        self._ck(self.lib.chemora_get_state_ghosted(self._h, out.ctypes.data_as(ctypes.c_void_p)))
        return out

    def enforce_constraints(self, state=None):
        """in place on a padded device state tensor (default: U)"""
        self._ck(self.lib.chemora_enforce_constraints(self._h, None if state is None else state.data_ptr()))

    def energy(self, state=None, field=False):
        """Sample-1 energy of a padded device state (default U): the grid sum, and the packed field if asked."""
        import torch
        total = ctypes.c_double()
        nx, ny, nz = self.dims
        eps = torch.empty((nz, ny, nx), dtype=torch.float64, device=self.device) if field else None
        self._ck(self.lib.chemora_energy(self._h, None if state is None else state.data_ptr(),
                                         None if eps is None else eps.data_ptr(), ctypes.byref(total)))
        return (total.value, eps) if field else total.value

    def set_variant(self, fused, tile_id):
        self._ck(self.lib.chemora_set_variant(self._h, int(fused), int(tile_id)))

    def get_variant(self):
        f, t = ctypes.c_int(), ctypes.c_int()
        self._ck(self.lib.chemora_get_variant(self._h, f, t))
        return f.value, t.value

    def autotune(self):
        f, t = ctypes.c_int(), ctypes.c_int()
        ms = (ctypes.c_float * (2 * NUM_TILES))()
        self._ck(self.lib.chemora_autotune(self._h, f, t, ms))
        return f.value, t.value, list(ms)

    def launch_count(self):
        return self.lib.chemora_launch_count(self._h)

    def kernel_info(self):
        r, l, s = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
        self._ck(self.lib.chemora_kernel_info(self._h, r, l, s))
        return dict(regs=r.value, local_bytes=l.value, smem_bytes=s.value)

    def timing(self, enable):
        self._ck(self.lib.chemora_timing(self._h, int(enable)))

    def timing_read(self):
        a, b, c, d = ctypes.c_double(), ctypes.c_long(), ctypes.c_double(), ctypes.c_long()
        self._ck(self.lib.chemora_timing_read(self._h, a, b, c, d))
        return dict(rhs_ms=a.value, rhs_launches=b.value, fill_ms=c.value, fill_launches=d.value)

    def measure_box_fill(self, tile_id):
        """ms of one fill-only launch of fused tile id `tile_id` (chemora_measure_box_fill)"""
        ms = ctypes.c_float()
        self._ck(self.lib.chemora_measure_box_fill(self._h, int(tile_id), ctypes.byref(ms)))
        return ms.value

    def measure_fp64_peak(self):
        v = ctypes.c_double()
        self._ck(self.lib.chemora_measure_fp64_peak(self._h, v))
        return v.value

    def destroy(self):
        if self._h:
            self.lib.chemora_destroy(self._h)
            self._h = ctypes.c_void_p()
            self._owned.clear()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
