"""ORACLE -- test infrastructure, NOT part of the product.

ctypes front end of oracle/rans_oracle.c (static order-0 rANS over the occupancy bytes; rules:
reading [R17], stated in the C file's header)."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "rans_oracle.c")
_LIB = os.path.join(_DIR, "librans_oracle.so")
_lib = None
BLOCK = 1024


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(["gcc", "-O1", "-shared", "-fPIC", "-o", _LIB, _SRC], check=True)
    return _LIB


def _L():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        u64, vp = ctypes.c_uint64, ctypes.c_void_p
        L.rans_oracle_model.restype = None
        L.rans_oracle_model.argtypes = [vp, u64, vp]
        L.rans_oracle_encode.restype = u64
        L.rans_oracle_encode.argtypes = [vp, u64, vp, vp, vp]
        L.rans_oracle_decode.restype = ctypes.c_int
        L.rans_oracle_decode.argtypes = [vp, u64, vp, vp, vp, u64]
        _lib = L
    return _lib


def model(data):
    d = np.ascontiguousarray(data, dtype=np.uint8)
    f = np.zeros(256, dtype=np.uint16)
    _L().rans_oracle_model(d.ctypes.data if d.size else None, d.size, f.ctypes.data)
    return f


def encode(data):
    """bytes -> (freq[256] uint16, nwords[nblk] uint16, payload uint8)."""
    d = np.ascontiguousarray(data, dtype=np.uint8)
    nblk = (d.size + BLOCK - 1) // BLOCK
    f = np.zeros(256, dtype=np.uint16)
    nw = np.zeros(max(nblk, 1), dtype=np.uint16)
    total = _L().rans_oracle_encode(d.ctypes.data if d.size else None, d.size, f.ctypes.data, nw.ctypes.data, None)
    payload = np.zeros(max(int(total), 1), dtype=np.uint8)
    _L().rans_oracle_encode(d.ctypes.data if d.size else None, d.size, f.ctypes.data, nw.ctypes.data, payload.ctypes.data)
    return f, nw[:nblk], payload[:int(total)]


def decode(payload, f, nwords, n):
    p = np.ascontiguousarray(payload, dtype=np.uint8)
    out = np.zeros(max(n, 1), dtype=np.uint8)
    bad = _L().rans_oracle_decode(p.ctypes.data if p.size else None, p.size, np.ascontiguousarray(f, np.uint16).ctypes.data,
                                  np.ascontiguousarray(nwords, np.uint16).ctypes.data, out.ctypes.data, n)
    return out[:n], bool(bad)
