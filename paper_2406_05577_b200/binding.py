"""Thin Python binding of the C-ABI in include/fftb.h (argument marshalling only).

Every step of the transform runs in the CUDA kernels behind ``libfftb.so``; PyTorch is used for
device memory and streams.  There is no CPU fallback: if the library has not been built, loading
fails with an ImportError that says how to build it.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_LIBPATH = _HERE / "libfftb.so"

FFTB_C64, FFTB_C128 = 0, 1
FFTB_SCALE_NONE, FFTB_SCALE_FORWARD = 0, 1
FFTB_FLAG_DENSE = 1
FFTB_FLAG_BATCH_FASTEST = 2
FFTB_TUNE_GENERIC_Z, FFTB_TUNE_GENERIC_PLANE, FFTB_TUNE_FUSED, FFTB_TUNE_NO_L2_HINTS, FFTB_TUNE_HOST_DEFER = 1, 2, 4, 8, 16
FFTB_OK, FFTB_EINVAL, FFTB_EUNSUPPORTED, FFTB_ENOMEM, FFTB_ECUDA, FFTB_ESTATE, FFTB_ETOOBIG = 0, -1, -2, -3, -4, -5, -6
FFTB_STATIC_SCRATCH_BYTES = 16 * 1024 * 1024  # the library-held device array fftb_inverse_static works in

# every symbol include/fftb.h declares
SYMBOLS = [
    "fftb_plan_create", "fftb_plan_create_tuned", "fftb_plan_create_explicit", "fftb_plan_create_explicit_tuned", "fftb_plan_info_get", "fftb_plan_get_map", "fftb_plan_bind",
    "fftb_inverse", "fftb_inverse_static", "fftb_forward", "fftb_apply_vloc",
    "fftb_inverse_host", "fftb_forward_host", "fftb_apply_vloc_host", "fftb_host_flush",
    "fftb_dense_embed", "fftb_dense_extract", "fftb_packed_transpose",
    "fftb_probe_fma", "fftb_probe_store_port", "fftb_plan_last_launches",
    "fftb_slab_plan_create", "fftb_slab_plan_info_get", "fftb_slab_plan_counts", "fftb_slab_plan_bind", "fftb_slab_plan_exchange_ptr",
    "fftb_slab_inverse_begin", "fftb_slab_inverse_end", "fftb_slab_forward_begin", "fftb_slab_forward_end", "fftb_slab_plan_destroy", "fftb_plan_profile", "fftb_plan_profile_read", "fftb_plan_destroy", "fftb_strerror",
]


class PlanDesc(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int32 * 3), ("cutoff", ctypes.c_int32 * 3), ("batch", ctypes.c_int32),
                ("dtype", ctypes.c_int32), ("scale", ctypes.c_int32), ("flags", ctypes.c_uint32)]


class PlanInfo(ctypes.Structure):
    _fields_ = [(k, ctypes.c_int64) for k in (
        "n_points", "n_sticks", "n_xocc", "device_bytes", "device_bytes_host", "chunk_bands",
        "min_bytes_per_band_dir", "workspace_offset", "pitch", "y_residues", "chunk_bands_fwd", "chunk_bands_vloc",
        "ring_bands", "lead_bands", "ring_tile_sticks", "ring_tile_elems", "ring_pair_pitch")]


class PlanTuning(ctypes.Structure):
    _fields_ = [("workspace_bytes", ctypes.c_int64), ("ring_bands", ctypes.c_int32), ("lead_bands", ctypes.c_int32),
                ("flags", ctypes.c_uint32), ("z_ctas", ctypes.c_uint32)]


class FftbError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        super().__init__(f"{what}: {strerror(code)} ({code})")


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not _LIBPATH.exists():
            raise ImportError(
                f"{_LIBPATH} not found: build it with `python -m paper_2406_05577_b200.build` "
                "(there is no CPU fallback)")
        L = ctypes.CDLL(str(_LIBPATH))
        vp, i32 = ctypes.c_void_p, ctypes.c_int
        L.fftb_plan_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(PlanDesc)]
        L.fftb_plan_create_tuned.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(PlanDesc), ctypes.POINTER(PlanTuning)]
        L.fftb_plan_create_explicit.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(PlanDesc), ctypes.c_int64, vp, vp, vp, vp]
        L.fftb_plan_create_explicit_tuned.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(PlanDesc), ctypes.c_int64, vp, vp, vp, vp,
                                                      ctypes.POINTER(PlanTuning)]
        L.fftb_plan_info_get.argtypes = [vp, ctypes.POINTER(PlanInfo)]
        L.fftb_plan_get_map.argtypes = [vp, vp, vp, vp, vp, vp]
        L.fftb_plan_bind.argtypes = [vp, vp, ctypes.c_size_t, vp]
        for name in ("fftb_inverse", "fftb_inverse_static", "fftb_forward", "fftb_inverse_host", "fftb_forward_host"):
            getattr(L, name).argtypes = [vp, vp, vp, i32, vp]
        for name in ("fftb_apply_vloc", "fftb_apply_vloc_host"):
            getattr(L, name).argtypes = [vp, vp, vp, vp, i32, vp]
        for name in ("fftb_dense_embed", "fftb_dense_extract"):
            getattr(L, name).argtypes = [vp, vp, vp, vp, i32, vp]
        L.fftb_host_flush.argtypes = [vp, vp]
        L.fftb_packed_transpose.argtypes = [vp, vp, vp, i32, i32, vp]
        L.fftb_probe_fma.argtypes = [i32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        L.fftb_probe_store_port.argtypes = [i32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        L.fftb_plan_last_launches.argtypes = [vp]
        L.fftb_plan_profile.argtypes = [vp, i32]
        L.fftb_plan_profile_read.argtypes = [vp, vp, vp]
        L.fftb_plan_destroy.argtypes = [vp]
        L.fftb_strerror.argtypes = [i32]
        L.fftb_strerror.restype = ctypes.c_char_p
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().fftb_strerror(code).decode()


def probe_fma(dtype="c128"):
    """-> (TFLOP/s, ms) of the register-only FMA probe on the current device (fftb_probe_fma)."""
    tf, ms = ctypes.c_double(), ctypes.c_double()
    _check(lib().fftb_probe_fma(FFTB_C128 if dtype == "c128" else FFTB_C64, ctypes.byref(tf), ctypes.byref(ms)), "fftb_probe_fma")
    return tf.value, ms.value


def probe_store_port(n_sms):
    """-> (bytes per clock per SM, aggregate GB/s) of n_sms SMs streaming 32-byte stores (fftb_probe_store_port)."""
    v, g = ctypes.c_double(), ctypes.c_double()
    _check(lib().fftb_probe_store_port(int(n_sms), ctypes.byref(v), ctypes.byref(g)), "fftb_probe_store_port")
    return v.value, g.value


def _check(rc, what):
    if rc != 0:
        raise FftbError(rc, what)


def _stream_ptr(stream=None):
    import torch

    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


class Plan:
    """fftb_plan_create / bind / execute / destroy.  Tensors are torch CUDA tensors (or pinned host
    tensors for the *_host calls); shapes follow include/fftb.h: packed (nb, S), cuboid (nb, N3, N2, N1)."""

    def __init__(self, n, cutoff=(0, 0, 0), batch=1, dtype="c128", scale="forward", dense=False, stick_map=None, tuning=None,
                 batch_fastest=False):
        """stick_map = (k1, k2, k3lo, len) int arrays: fftb_plan_create_explicit instead of a cut-off.
        tuning = dict(workspace_bytes=, ring_bands=, lead_bands=, flags=, z_ctas=): fftb_plan_create_tuned."""
        d = PlanDesc()
        d.n[:] = [int(x) for x in n]
        d.cutoff[:] = [int(x) for x in cutoff]
        d.batch = int(batch)
        d.dtype = FFTB_C128 if dtype == "c128" else FFTB_C64
        d.scale = FFTB_SCALE_FORWARD if scale == "forward" else FFTB_SCALE_NONE
        d.flags = (FFTB_FLAG_DENSE if dense else 0) | (FFTB_FLAG_BATCH_FASTEST if batch_fastest else 0)
        self.batch_fastest = bool(batch_fastest)
        self._h = ctypes.c_void_p()
        tu = None
        if tuning is not None:
            tu = PlanTuning()
            tu.workspace_bytes = int(tuning.get("workspace_bytes", 0))
            tu.ring_bands = int(tuning.get("ring_bands", 0))
            tu.lead_bands = int(tuning.get("lead_bands", 0))
            tu.flags = int(tuning.get("flags", 0))
            tu.z_ctas = int(tuning.get("z_ctas", 0))
        if stick_map is None and tu is not None:
            _check(lib().fftb_plan_create_tuned(ctypes.byref(self._h), ctypes.byref(d), ctypes.byref(tu)), "fftb_plan_create_tuned")
        elif stick_map is None:
            _check(lib().fftb_plan_create(ctypes.byref(self._h), ctypes.byref(d)), "fftb_plan_create")
        else:
            m = [np.ascontiguousarray(x, dtype=np.int32) for x in stick_map]
            assert len(m) == 4 and all(x.shape == m[0].shape and x.ndim == 1 for x in m)
            ptrs = [x.ctypes.data_as(ctypes.c_void_p) for x in m]
            if tu is None:
                _check(lib().fftb_plan_create_explicit(ctypes.byref(self._h), ctypes.byref(d), ctypes.c_int64(m[0].size), *ptrs),
                       "fftb_plan_create_explicit")
            else:
                _check(lib().fftb_plan_create_explicit_tuned(ctypes.byref(self._h), ctypes.byref(d), ctypes.c_int64(m[0].size), *ptrs,
                                                             ctypes.byref(tu)), "fftb_plan_create_explicit_tuned")
        self.n = tuple(int(x) for x in n)
        self.batch = int(batch)
        self.dtype = dtype
        self.dense = dense
        info = PlanInfo()
        _check(lib().fftb_plan_info_get(self._h, ctypes.byref(info)), "fftb_plan_info_get")
        self.info = {k: int(getattr(info, k)) for k, _ in PlanInfo._fields_}
        self.S = self.info["n_points"]
        self.mem = None

    # ---- host-side queries
    def get_map(self):
        ns = self.info["n_sticks"]
        m = {k: np.empty(ns, dtype=np.int32) for k in ("k1", "k2", "k3lo", "len")}
        m["off"] = np.empty(ns + 1, dtype=np.int64)
        _check(lib().fftb_plan_get_map(self._h, *[m[k].ctypes.data_as(ctypes.c_void_p)
                                                  for k in ("k1", "k2", "k3lo", "len", "off")]), "fftb_plan_get_map")
        return m

    def points(self):
        """(k1, k2, k3) of every packed point, expanded from the stick map."""
        m = self.get_map()
        rep = np.repeat(np.arange(len(m["k1"])), m["len"])
        k3 = m["k3lo"][rep] + (np.arange(self.S) - m["off"][:-1][rep]).astype(np.int32)
        return m["k1"][rep], m["k2"][rep], k3.astype(np.int32)

    # ---- device memory
    @property
    def torch_complex(self):
        import torch

        return torch.complex128 if self.dtype == "c128" else torch.complex64

    @property
    def torch_real(self):
        import torch

        return torch.float64 if self.dtype == "c128" else torch.float32

    def bind(self, mem=None, host_staging=False, device="cuda"):
        import torch

        need = self.info["device_bytes_host"] if host_staging else self.info["device_bytes"]
        if mem is None:
            mem = torch.empty(need, dtype=torch.uint8, device=device)
        assert mem.is_cuda and mem.dtype == torch.uint8 and mem.is_contiguous()
        _check(lib().fftb_plan_bind(self._h, ctypes.c_void_p(mem.data_ptr()), mem.numel(), _stream_ptr()), "fftb_plan_bind")
        self.mem = mem
        return self

    def _chk(self, t, shape, cuda=True, dtype=None):
        assert tuple(t.shape) == tuple(shape), (tuple(t.shape), tuple(shape))
        assert t.is_contiguous() and t.dtype == (dtype or self.torch_complex) and t.is_cuda == cuda
        return ctypes.c_void_p(t.data_ptr())

    def cuboid_shape(self, nb):
        return (nb, self.n[2], self.n[1], self.n[0])

    def packed_shape(self, nb):
        """(nb, S), or (S, nb) for a FFTB_FLAG_BATCH_FASTEST plan"""
        return (self.S, nb) if self.batch_fastest else (nb, self.S)

    def _nb(self, packed):
        return packed.shape[1] if self.batch_fastest else packed.shape[0]

    # ---- execute
    def inverse(self, packed, cuboid=None, stream=None):
        import torch

        nb = self._nb(packed)
        if cuboid is None:
            cuboid = torch.empty(self.cuboid_shape(nb), dtype=self.torch_complex, device=packed.device)
        _check(lib().fftb_inverse(self._h, self._chk(packed, self.packed_shape(nb)), self._chk(cuboid, self.cuboid_shape(nb)),
                                  nb, _stream_ptr(stream)), "fftb_inverse")
        return cuboid

    def inverse_static(self, packed, cuboid, stream=None):
        """fftb_inverse_static: no bind block; tables and intermediate in the library's static device array.  The caller
        passes the output too (this call allocates nothing)."""
        nb = self._nb(packed)
        _check(lib().fftb_inverse_static(self._h, self._chk(packed, self.packed_shape(nb)), self._chk(cuboid, self.cuboid_shape(nb)),
                                         nb, _stream_ptr(stream)), "fftb_inverse_static")
        return cuboid

    def forward(self, cuboid, packed=None, stream=None):
        import torch

        nb = cuboid.shape[0]
        if packed is None:
            packed = torch.empty(self.packed_shape(nb), dtype=self.torch_complex, device=cuboid.device)
        _check(lib().fftb_forward(self._h, self._chk(cuboid, self.cuboid_shape(nb)), self._chk(packed, self.packed_shape(nb)),
                                  nb, _stream_ptr(stream)), "fftb_forward")
        return packed

    def apply_vloc(self, packed_in, vloc, packed_out=None, stream=None):
        import torch

        nb = self._nb(packed_in)
        if packed_out is None:
            packed_out = torch.empty_like(packed_in)
        _check(lib().fftb_apply_vloc(self._h, self._chk(packed_in, self.packed_shape(nb)), self._chk(packed_out, self.packed_shape(nb)),
                                     self._chk(vloc, (self.n[2], self.n[1], self.n[0]), dtype=self.torch_real),
                                     nb, _stream_ptr(stream)), "fftb_apply_vloc")
        return packed_out

    def inverse_host(self, h_packed, cuboid, stream=None):
        nb = self._nb(h_packed)
        _check(lib().fftb_inverse_host(self._h, self._chk(h_packed, self.packed_shape(nb), cuda=False),
                                       self._chk(cuboid, self.cuboid_shape(nb)), nb, _stream_ptr(stream)), "fftb_inverse_host")
        return cuboid

    def forward_host(self, cuboid, h_packed, stream=None):
        nb = cuboid.shape[0]
        _check(lib().fftb_forward_host(self._h, self._chk(cuboid, self.cuboid_shape(nb)),
                                       self._chk(h_packed, self.packed_shape(nb), cuda=False), nb, _stream_ptr(stream)), "fftb_forward_host")
        return h_packed

    def apply_vloc_host(self, h_in, h_out, vloc, stream=None):
        nb = self._nb(h_in)
        _check(lib().fftb_apply_vloc_host(self._h, self._chk(h_in, self.packed_shape(nb), cuda=False),
                                          self._chk(h_out, self.packed_shape(nb), cuda=False),
                                          self._chk(vloc, (self.n[2], self.n[1], self.n[0]), dtype=self.torch_real),
                                          nb, _stream_ptr(stream)), "fftb_apply_vloc_host")
        return h_out

    def host_flush(self, stream=None):
        """FFTB_TUNE_HOST_DEFER plans: make the stream wait for the device-to-host copies of all *_host calls so far."""
        _check(lib().fftb_host_flush(self._h, _stream_ptr(stream)), "fftb_host_flush")

    def dense_embed(self, dense_plan, packed, packed_dense=None, stream=None):
        import torch

        nb = packed.shape[0]
        if packed_dense is None:
            packed_dense = torch.empty((nb, dense_plan.S), dtype=self.torch_complex, device=packed.device)
        _check(lib().fftb_dense_embed(self._h, dense_plan._h, self._chk(packed, (nb, self.S)),
                                      dense_plan._chk(packed_dense, (nb, dense_plan.S)), nb, _stream_ptr(stream)), "fftb_dense_embed")
        return packed_dense

    def dense_extract(self, dense_plan, packed_dense, packed=None, stream=None):
        import torch

        nb = packed_dense.shape[0]
        if packed is None:
            packed = torch.empty((nb, self.S), dtype=self.torch_complex, device=packed_dense.device)
        _check(lib().fftb_dense_extract(self._h, dense_plan._h, dense_plan._chk(packed_dense, (nb, dense_plan.S)),
                                        self._chk(packed, (nb, self.S)), nb, _stream_ptr(stream)), "fftb_dense_extract")
        return packed

    def packed_to_band_slowest(self, packed_sb, out=None, stream=None):
        """[S][nb] (the paper's batch-fastest order) -> [nb][S] (this library's order)."""
        import torch

        nb = packed_sb.shape[1]
        if out is None:
            out = torch.empty((nb, self.S), dtype=self.torch_complex, device=packed_sb.device)
        _check(lib().fftb_packed_transpose(self._h, self._chk(packed_sb, (self.S, nb)), self._chk(out, (nb, self.S)), nb, 1,
                                           _stream_ptr(stream)), "fftb_packed_transpose")
        return out

    def packed_to_band_fastest(self, packed_bs, out=None, stream=None):
        """[nb][S] -> [S][nb]."""
        import torch

        nb = packed_bs.shape[0]
        if out is None:
            out = torch.empty((self.S, nb), dtype=self.torch_complex, device=packed_bs.device)
        _check(lib().fftb_packed_transpose(self._h, self._chk(packed_bs, (nb, self.S)), self._chk(out, (self.S, nb)), nb, 0,
                                           _stream_ptr(stream)), "fftb_packed_transpose")
        return out

    def last_launches(self) -> int:
        return int(lib().fftb_plan_last_launches(self._h))

    KERNEL_KINDS = ("zpass_inv", "plane_inv", "plane_fwd", "zpass_fwd", "plane_vloc", "fused_inv", "fused_fwd")

    def profile(self, enable: bool):
        _check(lib().fftb_plan_profile(self._h, int(bool(enable))), "fftb_plan_profile")

    def profile_read(self):
        """-> {kernel kind: (total ms, launches)} since profiling was enabled / last read."""
        ms = np.zeros(len(self.KERNEL_KINDS), dtype=np.float64)
        cnt = np.zeros(len(self.KERNEL_KINDS), dtype=np.int64)
        _check(lib().fftb_plan_profile_read(self._h, ms.ctypes.data_as(ctypes.c_void_p),
                                            cnt.ctypes.data_as(ctypes.c_void_p)), "fftb_plan_profile_read")
        return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(self.KERNEL_KINDS)}

    def destroy(self):
        if self._h:
            lib().fftb_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
