"""ORACLE -- test infrastructure, NOT part of the product.

ctypes front end of oracle/rlgr_oracle.c (the block-parallel RLGR coder of PAPER.md:L257, L803; rules: reading [R14],
stated in the C file's header).  Only tests/, __graft_entry__ and bench.py's oracle legs may import this."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "rlgr_oracle.c")
_LIB = os.path.join(_DIR, "librlgr_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(["gcc", "-O1", "-shared", "-fPIC", "-o", _LIB, _SRC], check=True)
    return _LIB


def _L():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        u64, u32, vp = ctypes.c_uint64, ctypes.c_uint32, ctypes.c_void_p
        L.rlgr_oracle_encode_block.restype = u64
        L.rlgr_oracle_encode_block.argtypes = [vp, u64, u64, vp]
        L.rlgr_oracle_decode_block.restype = ctypes.c_int
        L.rlgr_oracle_decode_block.argtypes = [vp, u64, vp, u64, u64]
        L.rlgr_oracle_encode.restype = u64
        L.rlgr_oracle_encode.argtypes = [vp, u64, u32, u32, vp, vp]
        L.rlgr_oracle_decode.restype = ctypes.c_int
        L.rlgr_oracle_decode.argtypes = [vp, vp, u64, u32, u32, vp]
        _lib = L
    return _lib


def encode_block(x) -> tuple[bytes, int]:
    """One block of coefficients -> (stream bytes, padded bit length)."""
    x = np.ascontiguousarray(x, dtype=np.int32)
    bits = _L().rlgr_oracle_encode_block(x.ctypes.data, x.size, 1, None)
    out = np.zeros(bits // 8, dtype=np.uint8)
    _L().rlgr_oracle_encode_block(x.ctypes.data, x.size, 1, out.ctypes.data)
    return out.tobytes(), int(bits)


def decode_block(stream: bytes, n: int):
    buf = np.frombuffer(stream, dtype=np.uint8).copy()
    x = np.zeros(n, dtype=np.int32)
    bad = _L().rlgr_oracle_decode_block(buf.ctypes.data, buf.size * 8, x.ctypes.data, n, 1)
    return x, bool(bad)


def encode(q, block: int):
    """n x C int32 coefficient tensor -> (block_bits[nblk * C] uint32, stream uint8)."""
    q = np.ascontiguousarray(q, dtype=np.int32)
    n, C = q.shape
    nblk = (n + block - 1) // block
    bits = np.zeros(nblk * C, dtype=np.uint32)
    total = _L().rlgr_oracle_encode(q.ctypes.data, n, C, block, bits.ctypes.data, None)
    stream = np.zeros(max(int(total), 1), dtype=np.uint8)
    _L().rlgr_oracle_encode(q.ctypes.data, n, C, block, bits.ctypes.data, stream.ctypes.data)
    return bits, stream[:int(total)]


def decode(stream, block_bits, n: int, C: int, block: int):
    stream = np.ascontiguousarray(stream, dtype=np.uint8)
    bits = np.ascontiguousarray(block_bits, dtype=np.uint32)
    q = np.zeros((n, C), dtype=np.int32)
    bad = _L().rlgr_oracle_decode(stream.ctypes.data if stream.size else None, bits.ctypes.data, n, C, block, q.ctypes.data)
    return q, bool(bad)
