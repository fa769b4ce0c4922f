"""CPU oracle for the collection BWT -- TEST INFRASTRUCTURE, not product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It never imports ``paper_1401_7457_b200`` and the product never
imports it.  The arithmetic lives in ``cx_oracle.c`` (plain C, the definition of);
this file only compiles it with gcc and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cx_oracle.c")
_LIB = os.path.join(_HERE, "libcx_oracle.so")

OK, BAD_BASE, NOMEM, ARG, SMALL_BUFFER = 0, -1, -2, -3, -4


class OracleError(RuntimeError):
    def __init__(self, code: int):
        super().__init__(f"cx_oracle error {code}")
        self.code = code


def build(force: bool = False) -> str:
    """Compile ``cx_oracle.c`` -> ``libcx_oracle.so`` (gcc -O2) if missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=gnu11", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u8p, u64p = ctypes.POINTER(ctypes.c_uint8), ctypes.POINTER(ctypes.c_uint64)
        lib.cx_oracle_bwt.argtypes = [u8p, u64p, ctypes.c_uint64, u8p, u64p]
        lib.cx_oracle_bwt.restype = ctypes.c_int
        lib.cx_oracle_bwt_with_prefix.argtypes = [u8p, u64p, ctypes.c_uint64, u8p, ctypes.c_uint64, u8p,
                                                  ctypes.c_uint64, u64p, u64p]
        lib.cx_oracle_bwt_with_prefix.restype = ctypes.c_int
        lib.cx_oracle_bwt_of_listed.argtypes = [u8p, u64p, ctypes.c_uint64, u64p, ctypes.c_uint64, u8p]
        lib.cx_oracle_bwt_of_listed.restype = ctypes.c_int
        _lib = lib
    return _lib


def _ptr(a: np.ndarray, ctype):
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def _prep(ascii_: np.ndarray, offsets: np.ndarray):
    text = np.ascontiguousarray(ascii_, dtype=np.uint8)
    off = np.ascontiguousarray(offsets, dtype=np.uint64)
    if text.size == 0:
        text = np.zeros(1, dtype=np.uint8)     # valid pointer for an empty text
    return text, off


def bwt(ascii_: np.ndarray, offsets: np.ndarray, return_order: bool = False):
    """B_R of PAPER.md:55 as ``uint8[N]`` over ``$ACGT``; optionally the sorted (read, pos) list."""
    text, off = _prep(ascii_, offsets)
    n = int(off.shape[0] - 1) if off.shape[0] else 0
    N = (int(off[-1]) + n) if n else 0
    out = np.empty(max(N, 1), dtype=np.uint8)
    order = np.empty((max(N, 1), 2), dtype=np.uint64) if return_order else None
    rc = _load().cx_oracle_bwt(_ptr(text, ctypes.c_uint8), _ptr(off, ctypes.c_uint64), n,
                               _ptr(out, ctypes.c_uint8),
                               _ptr(order, ctypes.c_uint64) if return_order else None)
    if rc:
        raise OracleError(rc)
    return (out[:N], order[:N]) if return_order else out[:N]


def bwt_with_prefix(ascii_: np.ndarray, offsets: np.ndarray, prefix: str):
    """Range-restricted oracle: (slice_offset, slice) for the suffixes that begin with ``prefix``."""
    text, off = _prep(ascii_, offsets)
    n = int(off.shape[0] - 1) if off.shape[0] else 0
    N = (int(off[-1]) + n) if n else 0
    p = np.frombuffer(prefix.encode("ascii"), dtype=np.uint8).copy() if prefix else np.zeros(1, np.uint8)
    so, sl = ctypes.c_uint64(0), ctypes.c_uint64(0)
    lib = _load()
    out = np.empty(max(N, 1), dtype=np.uint8)       # capacity N: one call (pages stay untouched)
    rc = lib.cx_oracle_bwt_with_prefix(_ptr(text, ctypes.c_uint8), _ptr(off, ctypes.c_uint64), n,
                                       _ptr(p, ctypes.c_uint8), len(prefix), _ptr(out, ctypes.c_uint8),
                                       out.shape[0], ctypes.byref(so), ctypes.byref(sl))
    if rc:
        raise OracleError(rc)
    assert int(so.value) + int(sl.value) <= N
    return int(so.value), out[:int(sl.value)].copy()


def bwt_of_listed(ascii_: np.ndarray, offsets: np.ndarray, listed: np.ndarray):
    """Sort the listed suffixes ((k, 2) array of (read, pos)) with the definition's comparator and return their
    preceding symbols in that order, plus the sorted list."""
    text, off = _prep(ascii_, offsets)
    n = int(off.shape[0] - 1) if off.shape[0] else 0
    lst = np.ascontiguousarray(listed, dtype=np.uint64).reshape(-1, 2).copy()
    out = np.empty(max(lst.shape[0], 1), dtype=np.uint8)
    rc = _load().cx_oracle_bwt_of_listed(_ptr(text, ctypes.c_uint8), _ptr(off, ctypes.c_uint64), n,
                                         _ptr(lst, ctypes.c_uint64), lst.shape[0], _ptr(out, ctypes.c_uint8))
    if rc:
        raise OracleError(rc)
    return out[:lst.shape[0]], lst


def bwt_of_strings(reads: list[str]) -> str:
    """Convenience for tiny cases: list of strings -> BWT string."""
    lens = np.array([len(r) for r in reads], dtype=np.uint64)
    off = np.zeros(len(reads) + 1, dtype=np.uint64)
    np.cumsum(lens, out=off[1:])
    text = np.frombuffer("".join(reads).encode("ascii"), dtype=np.uint8).copy()
    return bwt(text, off).tobytes().decode("ascii")
