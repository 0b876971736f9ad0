"""Thin ctypes binding over libgsnfs.so (C ABI: include/gsnfs.h).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.  PyTorch
supplies device memory (tensors) and the stream.  There is no CPU fallback -- if the library is
missing or a CUDA device is absent, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, c_char_p, c_float, c_int, c_uint32, c_uint64, c_void_p

import numpy as np
import torch

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libgsnfs.so")
_lib = None

GSNFS_OK = 0
GSNFS_E_INVALID_ARGUMENT = -1
GSNFS_E_CAPACITY = -2
GSNFS_E_CUDA = -3
GSNFS_E_CORRUPT_STREAM = -4
GSNFS_MAX_DEPTH = 21
GSNFS_MAX_CHANNELS = 208


class GsnfsQuant(ctypes.Structure):
    _fields_ = [("dz_round", c_float), ("recon_bias", c_float)]


class GsnfsCounts(ctypes.Structure):
    _fields_ = [("n_voxels", c_uint32), ("occ_bytes", c_uint32), ("status", c_uint32), ("reserved", c_uint32)]


class GsnfsFrameDesc(ctypes.Structure):
    _fields_ = [("depth", c_uint32), ("channels", c_uint32), ("n_voxels", c_uint32), ("occ_bytes", c_uint32),
                ("rlgr_block", c_uint32), ("flags", c_uint32), ("bbox_min", c_float * 3), ("bbox_max", c_float * 3),
                ("dz_round", c_float), ("recon_bias", c_float)]


class GsnfsSection(ctypes.Structure):
    _fields_ = [("id", c_uint32), ("reserved", c_uint32), ("data", c_void_p), ("bytes", c_uint64)]


SEC_LEVEL_SIZES, SEC_QSTEP, SEC_KLT, SEC_OCC_RAW, SEC_OCC_FREQ, SEC_OCC_NWORDS, SEC_OCC_PAYLOAD, SEC_WEIGHTS, SEC_COEF_BITS, \
    SEC_COEF_STREAM = range(1, 11)
GSNFS_MAX_SECTIONS = 16


class GsnfsError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        super().__init__(f"{where}: {lib().gsnfs_strerror(status).decode()} ({status}) {detail}")


_SIGNATURES = {
    "gsnfs_create": (c_int, [POINTER(c_void_p), c_int, c_uint64, c_int, c_int]),
    "gsnfs_destroy": (None, [c_void_p]),
    "gsnfs_strerror": (c_char_p, [c_int]),
    "gsnfs_last_error": (c_char_p, [c_void_p]),
    "gsnfs_version": (c_char_p, []),
    "gsnfs_poll_status": (c_int, [c_void_p]),
    "gsnfs_launch_count": (c_uint64, [c_void_p]),
    "gsnfs_occ_capacity": (c_uint64, [c_uint64, c_int]),
    "gsnfs_profile_start": (c_int, [c_void_p, c_int]),
    "gsnfs_profile_stop": (c_int, [c_void_p, c_char_p, c_uint64]),
    "gsnfs_octree_encode": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, POINTER(c_float), POINTER(c_float),
                                    c_int, c_void_p, c_uint64, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "gsnfs_voxel_merge": (c_int, [c_void_p, c_void_p, c_void_p, c_int, c_uint64, c_void_p, c_void_p, c_void_p,
                                  c_void_p, c_void_p]),
    "gsnfs_octree_decode": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, POINTER(c_uint32), c_int, c_void_p,
                                    c_void_p, c_void_p]),
    "gsnfs_raht_forward": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_int, c_void_p,
                                   c_int, POINTER(c_float), POINTER(GsnfsQuant), c_void_p, c_void_p]),
    "gsnfs_merge_raht_forward": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_int, c_void_p,
                                         c_int, POINTER(c_float), POINTER(GsnfsQuant), c_void_p, c_void_p, c_void_p]),
    "gsnfs_raht_inverse": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_int, c_void_p,
                                   c_void_p, c_int, POINTER(c_float), POINTER(GsnfsQuant), c_void_p]),
    "gsnfs_quantize": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_int, POINTER(c_float),
                               POINTER(GsnfsQuant), c_void_p]),
    "gsnfs_klt_floats": (c_uint64, [c_int]),
    "gsnfs_klt_fit": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_int, c_void_p]),
    "gsnfs_color_forward": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_int, c_void_p, c_void_p]),
    "gsnfs_color_inverse": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_int, c_void_p, c_void_p]),
    "gsnfs_rlgr_blocks": (c_uint64, [c_uint64, c_int, c_int]),
    "gsnfs_rlgr_capacity": (c_uint64, [c_uint64, c_int, c_int]),
    "gsnfs_rlgr_encode": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_int, c_int, c_void_p, c_void_p,
                                  c_uint64, c_void_p]),
    "gsnfs_rlgr_decode": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_uint64, c_int, c_int, c_void_p,
                                  c_void_p]),
    "gsnfs_rans_blocks": (c_uint64, [c_uint64]),
    "gsnfs_rans_capacity": (c_uint64, [c_uint64]),
    "gsnfs_rans_encode": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_void_p, c_void_p, c_void_p, c_uint64,
                                  c_void_p]),
    "gsnfs_rans_decode": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, c_void_p, c_void_p, c_uint64, c_void_p, c_void_p]),
    "gsnfs_rans_decode_static": (c_int, [c_void_p, c_void_p, c_uint64, c_void_p, c_void_p, c_uint64, c_void_p, c_void_p]),
    "gsnfs_container_size": (c_uint64, [POINTER(GsnfsSection), c_int]),
    "gsnfs_container_pack": (c_int, [POINTER(GsnfsFrameDesc), POINTER(GsnfsSection), c_int, c_void_p, c_uint64,
                                     POINTER(c_uint64)]),
    "gsnfs_container_unpack": (c_int, [c_void_p, c_uint64, POINTER(GsnfsFrameDesc), POINTER(GsnfsSection), c_int,
                                       POINTER(c_int)]),
    "gsnfs_frame_encode_host": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_uint64, c_int, POINTER(c_float),
                                        POINTER(c_float), c_int, POINTER(c_float), POINTER(GsnfsQuant), c_void_p,
                                        c_uint64, c_void_p, c_void_p, c_void_p, c_void_p]),
    "gsnfs_frame_decode_host": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, POINTER(c_uint32), c_int, c_void_p,
                                        c_void_p, c_int, POINTER(c_float), POINTER(GsnfsQuant), c_void_p, c_void_p,
                                        c_void_p]),
    "gsnfs_frame_encode_host_packed": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_uint64, c_int, POINTER(c_float),
                                               POINTER(c_float), c_int, POINTER(c_float), POINTER(GsnfsQuant), c_int,
                                               c_void_p, c_uint64, c_void_p, c_void_p, c_void_p, c_void_p, c_uint64,
                                               c_void_p, c_void_p]),
    "gsnfs_frame_decode_host_packed": (c_int, [c_void_p, c_void_p, c_void_p, c_uint64, POINTER(c_uint32), c_int, c_void_p,
                                               c_void_p, c_void_p, c_uint64, c_int, c_int, POINTER(c_float),
                                               POINTER(GsnfsQuant), c_void_p, c_void_p, c_void_p]),
}


def lib_path() -> str:
    return _LIB_PATH


def lib():
    """Load libgsnfs.so (once).  Raises if it has not been built -- there is no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} not built: run `python -m paper_2606_05650_b200.build` "
                               "(nvcc, sm_100a).  gsnfs has no CPU fallback.")
        L = ctypes.CDLL(_LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def exported_symbols():
    return sorted(_SIGNATURES)


# ----------------------------------------------------------------------------- helpers
def _dptr(t, dtype=None, name="tensor"):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"{name} must have dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    return c_void_p(t.data_ptr())


def _hptr(t, dtype, name):
    """Host buffer (torch CPU tensor, ideally pinned)."""
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous CPU tensor of dtype {dtype}")
    return c_void_p(t.data_ptr())


def _f3(v):
    a = np.asarray(v, dtype=np.float32).reshape(3)
    return (c_float * 3)(*a.tolist())


def _farr(v, n):
    if v is None:
        return None
    a = np.ascontiguousarray(np.asarray(v, dtype=np.float32).reshape(-1))
    if a.shape[0] != n:
        raise ValueError(f"expected {n} per-channel steps, got {a.shape[0]}")
    return (c_float * n)(*a.tolist())


def _quant(q):
    if q is None:
        return None
    return ctypes.pointer(GsnfsQuant(float(q[0]), float(q[1])))


def _stream(stream):
    if stream is None:
        return c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, torch.cuda.Stream):
        return c_void_p(stream.cuda_stream)
    return c_void_p(int(stream))


def gsnfs_occ_capacity(n: int, depth: int) -> int:
    return int(lib().gsnfs_occ_capacity(int(n), int(depth)))


def gsnfs_version() -> str:
    return lib().gsnfs_version().decode()


class Context:
    """gsnfs_ctx: owns the library's device scratch for frames up to the given sizes."""

    def __init__(self, max_points: int, max_channels: int = 56, max_depth: int = GSNFS_MAX_DEPTH, device: int = 0):
        if not torch.cuda.is_available():
            raise RuntimeError("gsnfs needs a CUDA device (sm_100a); there is no CPU fallback")
        h = c_void_p()
        rc = lib().gsnfs_create(ctypes.byref(h), int(device), int(max_points), int(max_channels), int(max_depth))
        if rc != GSNFS_OK:
            raise GsnfsError(rc, "gsnfs_create")
        self.handle = h
        self.device = int(device)
        self.max_points = int(max_points)
        self.max_channels = int(max_channels)
        self.max_depth = int(max_depth)

    def close(self):
        if getattr(self, "handle", None):
            lib().gsnfs_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def poll_status(self) -> int:
        """GSNFS_OK, or GSNFS_E_CAPACITY once if a kernel of this context reported a scratch overflow."""
        return int(lib().gsnfs_poll_status(self.handle))

    def launch_count(self) -> int:
        return int(lib().gsnfs_launch_count(self.handle))

    def profile_start(self, max_records: int = 4096):
        self._check(lib().gsnfs_profile_start(self.handle, int(max_records)), "gsnfs_profile_start")

    def profile_stop(self):
        """-> {kernel name: (launches, total_ms)}; synchronises the device."""
        buf = ctypes.create_string_buffer(1 << 14)
        self._check(lib().gsnfs_profile_stop(self.handle, buf, len(buf)), "gsnfs_profile_stop")
        out = {}
        for line in buf.value.decode().splitlines():
            name, cnt, ms = line.split()
            out[name] = (int(cnt), float(ms))
        return out

    def _check(self, rc, where):
        if rc != GSNFS_OK:
            raise GsnfsError(rc, where, lib().gsnfs_last_error(self.handle).decode() if rc == GSNFS_E_CUDA else "")


# ----------------------------------------------------------------------------- the ABI calls
def gsnfs_octree_encode(ctx: Context, d_xyz, n, bbox_min, bbox_max, depth, d_occ, d_level_sizes, d_perm,
                        d_voxel_keys, d_voxel_start, d_counts, stream=None):
    rc = lib().gsnfs_octree_encode(
        ctx.handle, _stream(stream), _dptr(d_xyz, torch.float32, "d_xyz"), int(n), _f3(bbox_min), _f3(bbox_max),
        int(depth), _dptr(d_occ, torch.uint8, "d_occ"), int(d_occ.numel()),
        _dptr(d_level_sizes, torch.int32, "d_level_sizes"), _dptr(d_perm, torch.int32, "d_perm"),
        _dptr(d_voxel_keys, torch.int64, "d_voxel_keys"), _dptr(d_voxel_start, torch.int32, "d_voxel_start"),
        _dptr(d_counts, torch.int32, "d_counts"))
    ctx._check(rc, "gsnfs_octree_encode")


def gsnfs_voxel_merge(ctx: Context, d_attr, channels, n, d_perm, d_voxel_start, d_counts, d_merged, d_weights,
                      stream=None):
    rc = lib().gsnfs_voxel_merge(
        ctx.handle, _stream(stream), _dptr(d_attr, torch.float32, "d_attr"), int(channels), int(n),
        _dptr(d_perm, torch.int32, "d_perm"), _dptr(d_voxel_start, torch.int32, "d_voxel_start"),
        _dptr(d_counts, torch.int32, "d_counts"), _dptr(d_merged, torch.float32, "d_merged"),
        _dptr(d_weights, torch.int32, "d_weights"))
    ctx._check(rc, "gsnfs_voxel_merge")


def gsnfs_octree_decode(ctx: Context, d_occ, occ_bytes, level_sizes, depth, d_voxel_xyz, d_voxel_keys, d_counts,
                        stream=None):
    ls = np.ascontiguousarray(np.asarray(level_sizes, dtype=np.uint32).reshape(-1))
    if ls.shape[0] != depth + 1:
        raise ValueError("level_sizes must have depth+1 entries")
    arr = (c_uint32 * (depth + 1))(*ls.tolist())
    rc = lib().gsnfs_octree_decode(
        ctx.handle, _stream(stream), _dptr(d_occ, torch.uint8, "d_occ"), int(occ_bytes), arr, int(depth),
        _dptr(d_voxel_xyz, torch.int32, "d_voxel_xyz"), _dptr(d_voxel_keys, torch.int64, "d_voxel_keys"),
        _dptr(d_counts, torch.int32, "d_counts"))
    ctx._check(rc, "gsnfs_octree_decode")


def gsnfs_raht_forward(ctx: Context, d_voxel_keys, d_weights, n_voxels, d_counts, depth, d_attr, channels, qstep,
                       quant, d_qcoeff, d_coeff, stream=None):
    rc = lib().gsnfs_raht_forward(
        ctx.handle, _stream(stream), _dptr(d_voxel_keys, torch.int64, "d_voxel_keys"),
        _dptr(d_weights, torch.int32, "d_weights"), int(n_voxels), _dptr(d_counts, torch.int32, "d_counts"),
        int(depth), _dptr(d_attr, torch.float32, "d_attr"), int(channels), _farr(qstep, channels), _quant(quant),
        _dptr(d_qcoeff, torch.int32, "d_qcoeff"), _dptr(d_coeff, torch.float32, "d_coeff"))
    ctx._check(rc, "gsnfs_raht_forward")


def gsnfs_merge_raht_forward(ctx: Context, d_voxel_keys, d_perm, d_voxel_start, n, d_counts, depth, d_attr, channels, qstep,
                             quant, d_weights_out, d_qcoeff, d_coeff, stream=None):
    rc = lib().gsnfs_merge_raht_forward(
        ctx.handle, _stream(stream), _dptr(d_voxel_keys, torch.int64, "d_voxel_keys"), _dptr(d_perm, torch.int32, "d_perm"),
        _dptr(d_voxel_start, torch.int32, "d_voxel_start"), int(n), _dptr(d_counts, torch.int32, "d_counts"), int(depth),
        _dptr(d_attr, torch.float32, "d_attr"), int(channels), _farr(qstep, channels), _quant(quant),
        _dptr(d_weights_out, torch.int32, "d_weights_out"), _dptr(d_qcoeff, torch.int32, "d_qcoeff"),
        _dptr(d_coeff, torch.float32, "d_coeff"))
    ctx._check(rc, "gsnfs_merge_raht_forward")


def gsnfs_quantize(ctx: Context, d_coeff, n_rows, d_counts, channels, qstep, quant, d_qcoeff, stream=None):
    rc = lib().gsnfs_quantize(
        ctx.handle, _stream(stream), _dptr(d_coeff, torch.float32, "d_coeff"), int(n_rows),
        _dptr(d_counts, torch.int32, "d_counts"), int(channels), _farr(qstep, channels), _quant(quant),
        _dptr(d_qcoeff, torch.int32, "d_qcoeff"))
    ctx._check(rc, "gsnfs_quantize")


def gsnfs_raht_inverse(ctx: Context, d_voxel_keys, d_weights, n_voxels, d_counts, depth, d_qcoeff, d_coeff, channels,
                       qstep, quant, d_attr_out, stream=None):
    rc = lib().gsnfs_raht_inverse(
        ctx.handle, _stream(stream), _dptr(d_voxel_keys, torch.int64, "d_voxel_keys"),
        _dptr(d_weights, torch.int32, "d_weights"), int(n_voxels), _dptr(d_counts, torch.int32, "d_counts"),
        int(depth), _dptr(d_qcoeff, torch.int32, "d_qcoeff"), _dptr(d_coeff, torch.float32, "d_coeff"),
        int(channels), _farr(qstep, channels), _quant(quant), _dptr(d_attr_out, torch.float32, "d_attr_out"))
    ctx._check(rc, "gsnfs_raht_inverse")


def gsnfs_klt_floats(channels: int) -> int:
    return int(lib().gsnfs_klt_floats(int(channels)))


def gsnfs_klt_fit(ctx: Context, d_attr, n_rows, d_counts, channels, d_klt, stream=None):
    rc = lib().gsnfs_klt_fit(ctx.handle, _stream(stream), _dptr(d_attr, torch.float32, "d_attr"), int(n_rows),
                             _dptr(d_counts, torch.int32, "d_counts"), int(channels), _dptr(d_klt, torch.float32, "d_klt"))
    ctx._check(rc, "gsnfs_klt_fit")


def gsnfs_color_forward(ctx: Context, d_attr, n_rows, d_counts, channels, d_klt, d_out, stream=None):
    rc = lib().gsnfs_color_forward(ctx.handle, _stream(stream), _dptr(d_attr, torch.float32, "d_attr"), int(n_rows),
                                   _dptr(d_counts, torch.int32, "d_counts"), int(channels),
                                   _dptr(d_klt, torch.float32, "d_klt"), _dptr(d_out, torch.float32, "d_out"))
    ctx._check(rc, "gsnfs_color_forward")


def gsnfs_color_inverse(ctx: Context, d_attr, n_rows, d_counts, channels, d_klt, d_out, stream=None):
    rc = lib().gsnfs_color_inverse(ctx.handle, _stream(stream), _dptr(d_attr, torch.float32, "d_attr"), int(n_rows),
                                   _dptr(d_counts, torch.int32, "d_counts"), int(channels),
                                   _dptr(d_klt, torch.float32, "d_klt"), _dptr(d_out, torch.float32, "d_out"))
    ctx._check(rc, "gsnfs_color_inverse")


def gsnfs_rlgr_blocks(n_rows: int, channels: int, block_size: int) -> int:
    return int(lib().gsnfs_rlgr_blocks(int(n_rows), int(channels), int(block_size)))


def gsnfs_rlgr_capacity(n_rows: int, channels: int, block_size: int) -> int:
    return int(lib().gsnfs_rlgr_capacity(int(n_rows), int(channels), int(block_size)))


def rlgr_info(d_info):
    """Host view of a device gsnfs_rlgr_info (an int64[2] tensor): (stream_bytes, n_blocks, status); synchronises."""
    v = d_info.cpu().numpy().view(np.uint64)
    return int(v[0]), int(v[1] & np.uint64(0xffffffff)), int(v[1] >> np.uint64(32))


def gsnfs_rlgr_encode(ctx: Context, d_qcoeff, n_rows, d_counts, channels, block_size, d_block_bits, d_stream, d_info,
                      stream=None):
    rc = lib().gsnfs_rlgr_encode(
        ctx.handle, _stream(stream), _dptr(d_qcoeff, torch.int32, "d_qcoeff"), int(n_rows),
        _dptr(d_counts, torch.int32, "d_counts"), int(channels), int(block_size),
        _dptr(d_block_bits, torch.int32, "d_block_bits"), _dptr(d_stream, torch.uint8, "d_stream"), int(d_stream.numel()),
        _dptr(d_info, torch.int64, "d_info"))
    ctx._check(rc, "gsnfs_rlgr_encode")


def gsnfs_rlgr_decode(ctx: Context, d_stream, stream_bytes, d_block_bits, n_rows, channels, block_size, d_qcoeff, d_info,
                      stream=None):
    rc = lib().gsnfs_rlgr_decode(
        ctx.handle, _stream(stream), _dptr(d_stream, torch.uint8, "d_stream"), int(stream_bytes),
        _dptr(d_block_bits, torch.int32, "d_block_bits"), int(n_rows), int(channels), int(block_size),
        _dptr(d_qcoeff, torch.int32, "d_qcoeff"), _dptr(d_info, torch.int64, "d_info"))
    ctx._check(rc, "gsnfs_rlgr_decode")


def gsnfs_rans_blocks(n: int) -> int:
    return int(lib().gsnfs_rans_blocks(int(n)))


def gsnfs_rans_capacity(n: int) -> int:
    return int(lib().gsnfs_rans_capacity(int(n)))


def gsnfs_rans_encode(ctx: Context, d_data, n, d_counts, d_freq, d_nwords, d_payload, d_info, stream=None):
    rc = lib().gsnfs_rans_encode(
        ctx.handle, _stream(stream), _dptr(d_data, torch.uint8, "d_data"), int(n), _dptr(d_counts, torch.int32, "d_counts"),
        _dptr(d_freq, torch.int16, "d_freq"), _dptr(d_nwords, torch.int16, "d_nwords"),
        _dptr(d_payload, torch.uint8, "d_payload"), int(d_payload.numel()), _dptr(d_info, torch.int64, "d_info"))
    ctx._check(rc, "gsnfs_rans_encode")


def gsnfs_rans_decode(ctx: Context, d_payload, payload_bytes, d_freq, d_nwords, n, d_out, d_info, stream=None):
    rc = lib().gsnfs_rans_decode(
        ctx.handle, _stream(stream), _dptr(d_payload, torch.uint8, "d_payload"), int(payload_bytes),
        _dptr(d_freq, torch.int16, "d_freq"), _dptr(d_nwords, torch.int16, "d_nwords"), int(n),
        _dptr(d_out, torch.uint8, "d_out"), _dptr(d_info, torch.int64, "d_info"))
    ctx._check(rc, "gsnfs_rans_decode")


GSNFS_RANS_STATIC_MAX_BYTES = 32 << 20


def gsnfs_rans_decode_static(d_payload, payload_bytes, d_freq, d_nwords, n, d_out, d_info, stream=None):
    """gsnfs_rans_decode for callers that may not allocate device memory (their own pool owns the GPU, a frozen memory
    budget, or a frame loop that cannot take cudaMalloc's device-wide synchronisation): no Context, no allocation; the
    block-offset table is a fixed 256 KB array inside the library.  n <= GSNFS_RANS_STATIC_MAX_BYTES, else GsnfsError
    (GSNFS_E_CAPACITY).  Runs on the current device; calls that overlap on the GPU race on the shared table; the first
    call on a device does a one-off address lookup and belongs before any stream capture (include/gsnfs.h)."""
    rc = lib().gsnfs_rans_decode_static(
        _stream(stream), _dptr(d_payload, torch.uint8, "d_payload"), int(payload_bytes),
        _dptr(d_freq, torch.int16, "d_freq"), _dptr(d_nwords, torch.int16, "d_nwords"), int(n),
        _dptr(d_out, torch.uint8, "d_out"), _dptr(d_info, torch.int64, "d_info"))
    if rc != GSNFS_OK:
        raise GsnfsError(rc, "gsnfs_rans_decode_static",
                         f"(n = {int(n)}, limit {GSNFS_RANS_STATIC_MAX_BYTES} bytes)" if rc == -2 else "")


def container_pack(desc: GsnfsFrameDesc, sections: dict) -> np.ndarray:
    """{section id: contiguous numpy array} -> one uint8 buffer (host only; marshalling of gsnfs_container_pack)."""
    arrs = {k: np.ascontiguousarray(v) for k, v in sections.items()}
    secs = (GsnfsSection * len(arrs))()
    for i, (k, a) in enumerate(arrs.items()):
        secs[i] = GsnfsSection(int(k), 0, a.ctypes.data if a.nbytes else None, a.nbytes)
    size = int(lib().gsnfs_container_size(secs, len(arrs)))
    out = np.zeros(size, dtype=np.uint8)
    written = c_uint64(0)
    rc = lib().gsnfs_container_pack(ctypes.byref(desc), secs, len(arrs), out.ctypes.data, size, ctypes.byref(written))
    if rc != GSNFS_OK:
        raise GsnfsError(rc, "gsnfs_container_pack")
    return out[:written.value]


def container_unpack(buf: np.ndarray):
    """uint8 buffer -> (GsnfsFrameDesc, {section id: uint8 view into buf}); raises GsnfsError on a damaged buffer."""
    buf = np.ascontiguousarray(buf, dtype=np.uint8)
    desc = GsnfsFrameDesc()
    secs = (GsnfsSection * GSNFS_MAX_SECTIONS)()
    n = c_int(0)
    rc = lib().gsnfs_container_unpack(buf.ctypes.data, buf.nbytes, ctypes.byref(desc), secs, GSNFS_MAX_SECTIONS, ctypes.byref(n))
    if rc != GSNFS_OK:
        raise GsnfsError(rc, "gsnfs_container_unpack")
    out = {}
    for i in range(n.value):
        off = (secs[i].data - buf.ctypes.data) if secs[i].bytes else 0
        out[int(secs[i].id)] = buf[off:off + secs[i].bytes]
    return desc, out


def gsnfs_frame_encode_host(ctx: Context, h_xyz, h_attr, n, channels, bbox_min, bbox_max, depth, qstep, quant,
                            h_occ, h_level_sizes, h_weights, h_qcoeff, h_counts, stream=None):
    rc = lib().gsnfs_frame_encode_host(
        ctx.handle, _stream(stream), _hptr(h_xyz, torch.float32, "h_xyz"), _hptr(h_attr, torch.float32, "h_attr"),
        int(n), int(channels), _f3(bbox_min), _f3(bbox_max), int(depth), _farr(qstep, channels), _quant(quant),
        _hptr(h_occ, torch.uint8, "h_occ"), int(h_occ.numel()), _hptr(h_level_sizes, torch.int32, "h_level_sizes"),
        _hptr(h_weights, torch.int32, "h_weights"), _hptr(h_qcoeff, torch.int32, "h_qcoeff"),
        _hptr(h_counts, torch.int32, "h_counts"))
    ctx._check(rc, "gsnfs_frame_encode_host")


def gsnfs_frame_decode_host(ctx: Context, h_occ, occ_bytes, level_sizes, depth, h_weights, h_qcoeff, channels, qstep,
                            quant, h_voxel_xyz, h_attr, h_counts, stream=None):
    ls = np.ascontiguousarray(np.asarray(level_sizes, dtype=np.uint32).reshape(-1))
    arr = (c_uint32 * (depth + 1))(*ls.tolist())
    rc = lib().gsnfs_frame_decode_host(
        ctx.handle, _stream(stream), _hptr(h_occ, torch.uint8, "h_occ"), int(occ_bytes), arr, int(depth),
        _hptr(h_weights, torch.int32, "h_weights"), _hptr(h_qcoeff, torch.int32, "h_qcoeff"), int(channels),
        _farr(qstep, channels), _quant(quant), _hptr(h_voxel_xyz, torch.int32, "h_voxel_xyz"),
        _hptr(h_attr, torch.float32, "h_attr"), _hptr(h_counts, torch.int32, "h_counts"))
    ctx._check(rc, "gsnfs_frame_decode_host")


def gsnfs_frame_encode_host_packed(ctx: Context, h_xyz, h_attr, n, channels, bbox_min, bbox_max, depth, qstep, quant,
                                   rlgr_block, h_occ, h_level_sizes, h_weights, h_block_bits, h_stream, h_counts, h_info,
                                   stream=None):
    rc = lib().gsnfs_frame_encode_host_packed(
        ctx.handle, _stream(stream), _hptr(h_xyz, torch.float32, "h_xyz"), _hptr(h_attr, torch.float32, "h_attr"),
        int(n), int(channels), _f3(bbox_min), _f3(bbox_max), int(depth), _farr(qstep, channels), _quant(quant),
        int(rlgr_block), _hptr(h_occ, torch.uint8, "h_occ"), int(h_occ.numel()),
        _hptr(h_level_sizes, torch.int32, "h_level_sizes"), _hptr(h_weights, torch.int32, "h_weights"),
        _hptr(h_block_bits, torch.int32, "h_block_bits"), _hptr(h_stream, torch.uint8, "h_stream"), int(h_stream.numel()),
        _hptr(h_counts, torch.int32, "h_counts"), _hptr(h_info, torch.int64, "h_info"))
    ctx._check(rc, "gsnfs_frame_encode_host_packed")


def gsnfs_frame_decode_host_packed(ctx: Context, h_occ, occ_bytes, level_sizes, depth, h_weights, h_block_bits, h_stream,
                                   stream_bytes, rlgr_block, channels, qstep, quant, h_voxel_xyz, h_attr, h_counts,
                                   stream=None):
    ls = np.ascontiguousarray(np.asarray(level_sizes, dtype=np.uint32).reshape(-1))
    arr = (c_uint32 * (depth + 1))(*ls.tolist())
    rc = lib().gsnfs_frame_decode_host_packed(
        ctx.handle, _stream(stream), _hptr(h_occ, torch.uint8, "h_occ"), int(occ_bytes), arr, int(depth),
        _hptr(h_weights, torch.int32, "h_weights"), _hptr(h_block_bits, torch.int32, "h_block_bits"),
        _hptr(h_stream, torch.uint8, "h_stream"), int(stream_bytes), int(rlgr_block), int(channels),
        _farr(qstep, channels), _quant(quant), _hptr(h_voxel_xyz, torch.int32, "h_voxel_xyz"),
        _hptr(h_attr, torch.float32, "h_attr"), _hptr(h_counts, torch.int32, "h_counts"))
    ctx._check(rc, "gsnfs_frame_decode_host_packed")


# ----------------------------------------------------------------------------- buffer bundle
class FrameBuffers:
    """Caller-owned device buffers for one frame (allocated by PyTorch; the library only fills them)."""

    def __init__(self, n: int, channels: int, depth: int, device="cuda:0"):
        dev = torch.device(device)
        self.n, self.channels, self.depth = int(n), int(channels), int(depth)
        cap = max(gsnfs_occ_capacity(n, depth), 16)
        n1 = max(n, 1)
        self.occ = torch.empty(cap, dtype=torch.uint8, device=dev)
        self.level_sizes = torch.zeros(depth + 1, dtype=torch.int32, device=dev)
        self.perm = torch.empty(n1, dtype=torch.int32, device=dev)
        self.voxel_keys = torch.empty(n1, dtype=torch.int64, device=dev)
        self.voxel_start = torch.empty(n1 + 1, dtype=torch.int32, device=dev)
        self.counts = torch.zeros(4, dtype=torch.int32, device=dev)
        self.merged = torch.empty((n1, channels), dtype=torch.float32, device=dev)
        self.weights = torch.empty(n1, dtype=torch.int32, device=dev)
        self.qcoeff = torch.empty((n1, channels), dtype=torch.int32, device=dev)
        # decoder side
        self.dec_xyz = torch.empty((n1, 3), dtype=torch.int32, device=dev)
        self.dec_keys = torch.empty(n1, dtype=torch.int64, device=dev)
        self.dec_counts = torch.zeros(4, dtype=torch.int32, device=dev)
        self.dec_attr = torch.empty((n1, channels), dtype=torch.float32, device=dev)


def encode_frame(ctx: Context, buf: FrameBuffers, d_xyz, d_attr, bbox_min, bbox_max, qstep, quant=None, stream=None,
                 fused=True):
    """The encoder's ABI calls chained on one stream with no host synchronisation.  fused=True uses
    gsnfs_merge_raht_forward (merge folded into the transform); fused=False the separate calls."""
    gsnfs_octree_encode(ctx, d_xyz, buf.n, bbox_min, bbox_max, buf.depth, buf.occ, buf.level_sizes, buf.perm,
                        buf.voxel_keys, buf.voxel_start, buf.counts, stream)
    if fused:
        gsnfs_merge_raht_forward(ctx, buf.voxel_keys, buf.perm, buf.voxel_start, buf.n, buf.counts, buf.depth, d_attr,
                                 buf.channels, qstep, quant, buf.weights, buf.qcoeff, None, stream)
        return
    gsnfs_voxel_merge(ctx, d_attr, buf.channels, buf.n, buf.perm, buf.voxel_start, buf.counts, buf.merged,
                      buf.weights, stream)
    gsnfs_raht_forward(ctx, buf.voxel_keys, buf.weights, buf.n, buf.counts, buf.depth, buf.merged, buf.channels,
                       qstep, quant, buf.qcoeff, None, stream)


def decode_frame(ctx: Context, buf: FrameBuffers, level_sizes, occ_bytes, qstep, quant=None, use_weights=True,
                 stream=None):
    """The decoder's two ABI calls.  level_sizes is the host-side stream header."""
    nv = int(level_sizes[buf.depth])
    gsnfs_octree_decode(ctx, buf.occ, occ_bytes, level_sizes, buf.depth, buf.dec_xyz, buf.dec_keys, buf.dec_counts,
                        stream)
    gsnfs_raht_inverse(ctx, buf.dec_keys, buf.weights if use_weights else None, nv, None, buf.depth, buf.qcoeff, None,
                       buf.channels, qstep, quant, buf.dec_attr, stream)
