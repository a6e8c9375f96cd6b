"""Slab-distributed transform over several GPUs: thin binding of the
fftb_slab_* calls of include/fftb.h plus the transport between ranks (torch.distributed all-to-all over NCCL).

Rank r owns the sticks of a contiguous range of occupied k1 columns -- the columns [packed_lo[r], packed_lo[r+1]) of every
band of the packed array -- and the z-planes [z_lo[r], z_lo[r+1]) of the cuboid.  Every arithmetic step and every pack /
unpack runs in the CUDA kernels behind libfftb.so; this module only marshals arguments and moves the staged blocks.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import binding as fb


class SlabInfo(ctypes.Structure):
    _fields_ = [(k, ctypes.c_int64) for k in ("n_points_local", "n_sticks_local", "planes_local", "device_bytes", "n_points", "n_sticks")]


_ready = False


def _lib():
    global _ready
    L = fb.lib()
    if not _ready:
        vp, i32 = ctypes.c_void_p, ctypes.c_int
        L.fftb_slab_plan_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(fb.PlanDesc), i32, i32]
        L.fftb_slab_plan_info_get.argtypes = [vp, ctypes.POINTER(SlabInfo)]
        L.fftb_slab_plan_counts.argtypes = [vp, vp, vp, vp]
        L.fftb_slab_plan_bind.argtypes = [vp, vp, ctypes.c_size_t, vp]
        L.fftb_slab_plan_exchange_ptr.argtypes = [vp, i32, ctypes.POINTER(vp)]
        L.fftb_slab_inverse_begin.argtypes = [vp, vp, vp, vp, i32, vp]
        L.fftb_slab_inverse_end.argtypes = [vp, vp, vp, i32, vp]
        L.fftb_slab_forward_begin.argtypes = [vp, vp, vp, vp, i32, vp]
        L.fftb_slab_forward_end.argtypes = [vp, vp, vp, i32, vp]
        L.fftb_slab_plan_destroy.argtypes = [vp]
        _ready = True
    return L


class SlabPlan:
    """One rank's share of a slab-distributed transform.  Tensors are torch CUDA tensors: packed_local (nb, n_points_local),
    cuboid_slab (nb, planes_local, N2, N1)."""

    def __init__(self, n, cutoff, batch, world, rank, dtype="c128", scale="forward"):
        d = fb.PlanDesc()
        d.n[:] = [int(x) for x in n]
        d.cutoff[:] = [int(x) for x in cutoff]
        d.batch = int(batch)
        d.dtype = fb.FFTB_C128 if dtype == "c128" else fb.FFTB_C64
        d.scale = fb.FFTB_SCALE_FORWARD if scale == "forward" else fb.FFTB_SCALE_NONE
        d.flags = 0
        self._h = ctypes.c_void_p()
        fb._check(_lib().fftb_slab_plan_create(ctypes.byref(self._h), ctypes.byref(d), int(world), int(rank)), "fftb_slab_plan_create")
        self.n, self.batch, self.world, self.rank, self.dtype = tuple(int(x) for x in n), int(batch), int(world), int(rank), dtype
        info = SlabInfo()
        fb._check(_lib().fftb_slab_plan_info_get(self._h, ctypes.byref(info)), "fftb_slab_plan_info_get")
        self.info = {k: int(getattr(info, k)) for k, _ in SlabInfo._fields_}
        self.stick_lo, self.packed_lo, self.z_lo = (np.zeros(world + 1, dtype=np.int64) for _ in range(3))
        fb._check(_lib().fftb_slab_plan_counts(self._h, *[a.ctypes.data_as(ctypes.c_void_p) for a in (self.stick_lo, self.packed_lo, self.z_lo)]),
                  "fftb_slab_plan_counts")
        self.mem = None

    # ---- sizes of the exchange, in elements, for nb bands: (send to every peer, receive from every peer)
    def counts(self, direction, nb):
        sticks, planes, r = np.diff(self.stick_lo), np.diff(self.z_lo), self.rank
        if direction == "inverse":   # rows = the receiver's planes, columns = the sender's sticks
            return [int(nb * planes[d] * sticks[r]) for d in range(self.world)], [int(nb * planes[r] * sticks[s]) for s in range(self.world)]
        return [int(nb * planes[r] * sticks[d]) for d in range(self.world)], [int(nb * planes[s] * sticks[r]) for s in range(self.world)]

    @property
    def torch_complex(self):
        import torch

        return torch.complex128 if self.dtype == "c128" else torch.complex64

    def bind(self, device="cuda"):
        import torch

        self.mem = torch.empty(self.info["device_bytes"], dtype=torch.uint8, device=device)
        fb._check(_lib().fftb_slab_plan_bind(self._h, ctypes.c_void_p(self.mem.data_ptr()), self.mem.numel(), fb._stream_ptr()), "fftb_slab_plan_bind")
        return self

    def exchange_ptr(self, which):
        p = ctypes.c_void_p()
        fb._check(_lib().fftb_slab_plan_exchange_ptr(self._h, int(which), ctypes.byref(p)), "fftb_slab_plan_exchange_ptr")
        return int(p.value)

    def cuboid_slab_shape(self, nb):
        return (nb, self.info["planes_local"], self.n[1], self.n[0])

    @staticmethod
    def _peers(ptrs):
        return None if ptrs is None else (ctypes.c_void_p * len(ptrs))(*[ctypes.c_void_p(int(x)) for x in ptrs])

    def _buf(self, t):
        return ctypes.c_void_p(0 if t is None else t.data_ptr())

    def inverse_begin(self, packed_local, send=None, peers=None, stream=None):
        nb = packed_local.shape[0]
        assert tuple(packed_local.shape) == (nb, self.info["n_points_local"]) and packed_local.is_contiguous()
        fb._check(_lib().fftb_slab_inverse_begin(self._h, self._buf(packed_local), self._peers(peers), self._buf(send), nb, fb._stream_ptr(stream)),
                  "fftb_slab_inverse_begin")

    def inverse_end(self, cuboid_slab, recv=None, stream=None):
        nb = cuboid_slab.shape[0]
        assert tuple(cuboid_slab.shape) == self.cuboid_slab_shape(nb) and cuboid_slab.is_contiguous()
        fb._check(_lib().fftb_slab_inverse_end(self._h, self._buf(recv), self._buf(cuboid_slab), nb, fb._stream_ptr(stream)), "fftb_slab_inverse_end")

    def forward_begin(self, cuboid_slab, send=None, peers=None, stream=None):
        nb = cuboid_slab.shape[0]
        assert tuple(cuboid_slab.shape) == self.cuboid_slab_shape(nb) and cuboid_slab.is_contiguous()
        fb._check(_lib().fftb_slab_forward_begin(self._h, self._buf(cuboid_slab), self._peers(peers), self._buf(send), nb, fb._stream_ptr(stream)),
                  "fftb_slab_forward_begin")

    def forward_end(self, packed_local, recv=None, stream=None):
        nb = packed_local.shape[0]
        assert tuple(packed_local.shape) == (nb, self.info["n_points_local"]) and packed_local.is_contiguous()
        fb._check(_lib().fftb_slab_forward_end(self._h, self._buf(recv), self._buf(packed_local), nb, fb._stream_ptr(stream)), "fftb_slab_forward_end")

    # ---- the whole distributed call: begin, all-to-all of the staged blocks over the default process group, end
    def _all_to_all(self, direction, nb, send):
        import torch
        import torch.distributed as dist

        s_cnt, r_cnt = self.counts(direction, nb)
        recv = torch.empty(sum(r_cnt), dtype=self.torch_complex, device=send.device)
        # complex tensors travel as their real views (2 reals per element)
        dist.all_to_all_single(torch.view_as_real(recv), torch.view_as_real(send), [c for c in r_cnt], [c for c in s_cnt])
        return recv

    def inverse(self, packed_local, cuboid_slab=None):
        import torch

        nb = packed_local.shape[0]
        if cuboid_slab is None:
            cuboid_slab = torch.empty(self.cuboid_slab_shape(nb), dtype=self.torch_complex, device=packed_local.device)
        send = torch.empty(sum(self.counts("inverse", nb)[0]), dtype=self.torch_complex, device=packed_local.device)
        self.inverse_begin(packed_local, send=send)
        self.inverse_end(cuboid_slab, recv=self._all_to_all("inverse", nb, send))
        return cuboid_slab

    def forward(self, cuboid_slab, packed_local=None):
        import torch

        nb = cuboid_slab.shape[0]
        if packed_local is None:
            packed_local = torch.empty((nb, self.info["n_points_local"]), dtype=self.torch_complex, device=cuboid_slab.device)
        send = torch.empty(sum(self.counts("forward", nb)[0]), dtype=self.torch_complex, device=cuboid_slab.device)
        self.forward_begin(cuboid_slab, send=send)
        self.forward_end(packed_local, recv=self._all_to_all("forward", nb, send))
        return packed_local

    def destroy(self):
        if self._h:
            _lib().fftb_slab_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
