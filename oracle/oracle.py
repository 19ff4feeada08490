"""ctypes front end of oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It holds no arithmetic of its own: every number is produced by
oracle.cpp (Eq. 4 of arxiv/paper_2606_08094).  Arrays are numpy,
bf16 is carried as uint16 bit patterns.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_SO = os.path.join(_HERE, "liboracle.so")
_FLAGS = ["-O3", "-march=native", "-fopenmp", "-fno-fast-math", "-ffp-contract=off",
          "-std=c++17", "-shared", "-fPIC"]
_lib = None


def build(force=False):
    """Compile oracle.cpp into oracle/liboracle.so with g++ (a second or two)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp%d" % os.getpid()
        subprocess.run(["g++", *_FLAGS, _SRC, "-o", tmp], check=True)
        os.replace(tmp, _SO)
    return _SO


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct)) if a is not None else None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_num_threads.restype = ctypes.c_int
        _lib.orc_pack_ref.restype = ctypes.c_long
    return _lib


def num_threads():
    return int(lib().orc_num_threads())


def _c(a, dt):
    a = np.ascontiguousarray(a)
    assert a.dtype == dt, (a.dtype, dt)
    return a


def bf16_to_f32(x_u16):
    x = _c(x_u16, np.uint16)
    out = np.empty(x.shape, np.float32)
    lib().orc_bf16_to_f32(_p(x, ctypes.c_uint16), ctypes.c_long(x.size), _p(out, ctypes.c_float))
    return out


def f32_to_bf16(x_f32):
    x = _c(x_f32, np.float32)
    out = np.empty(x.shape, np.uint16)
    lib().orc_f32_to_bf16(_p(x, ctypes.c_float), ctypes.c_long(x.size), _p(out, ctypes.c_uint16))
    return out


def act_quant(x_u16):
    """bf16 [M,K] -> (a int8 [M,K], alpha fp32 [M])   (Eq. 4 lines 1-2)."""
    x = _c(x_u16, np.uint16)
    M, K = x.shape
    a = np.empty((M, K), np.int8)
    alpha = np.empty((M,), np.float32)
    lib().orc_act_quant(_p(x, ctypes.c_uint16), M, K, _p(a, ctypes.c_int8), _p(alpha, ctypes.c_float))
    return a, alpha


def contract(a_i8, w_i8):
    """a [M,K] int8, w [N,K] int8 -> acc int32 [M,N]   (Eq. 4 line 3, the sum)."""
    a = _c(a_i8, np.int8)
    w = _c(w_i8, np.int8)
    M, K = a.shape
    N, K2 = w.shape
    assert K == K2
    acc = np.empty((M, N), np.int32)
    lib().orc_contract(_p(a, ctypes.c_int8), _p(w, ctypes.c_int8), M, N, K, _p(acc, ctypes.c_int32))
    return acc


def rescale(acc_i32, alpha_f32, beta):
    """-> (y fp32 [M,N], y64 float64 [M,N])   (Eq. 4 line 3, the scaling).  beta: scalar or [G]."""
    acc = _c(acc_i32, np.int32)
    alpha = _c(alpha_f32, np.float32)
    b = np.atleast_1d(np.asarray(beta, np.float32)).copy()
    M, N = acc.shape
    assert N % b.size == 0
    y32 = np.empty((M, N), np.float32)
    y64 = np.empty((M, N), np.float64)
    lib().orc_rescale(_p(acc, ctypes.c_int32), _p(alpha, ctypes.c_float), _p(b, ctypes.c_float),
                      int(b.size), M, N, _p(y32, ctypes.c_float), _p(y64, ctypes.c_double))
    return y32, y64


def ternary_linear(x_u16, w_i8, beta, want_y64=True):
    """Eq. 4 end to end.  Returns dict(a, alpha, acc, y32, ybf16, y64)."""
    x = _c(x_u16, np.uint16)
    w = _c(w_i8, np.int8)
    b = np.atleast_1d(np.asarray(beta, np.float32)).copy()
    M, K = x.shape
    N, K2 = w.shape
    assert K == K2 and N % b.size == 0
    a = np.empty((M, K), np.int8)
    alpha = np.empty((M,), np.float32)
    acc = np.empty((M, N), np.int32)
    y32 = np.empty((M, N), np.float32)
    ybf = np.empty((M, N), np.uint16)
    y64 = np.empty((M, N), np.float64) if want_y64 else None
    lib().orc_ternary_linear(_p(x, ctypes.c_uint16), _p(w, ctypes.c_int8), _p(b, ctypes.c_float),
                             int(b.size), M, N, K, _p(a, ctypes.c_int8), _p(alpha, ctypes.c_float),
                             _p(acc, ctypes.c_int32), _p(y32, ctypes.c_float),
                             _p(ybf, ctypes.c_uint16), _p(y64, ctypes.c_double))
    return dict(a=a, alpha=alpha, acc=acc, y32=y32, ybf16=ybf, y64=y64)


def pack_ref(w_i8):
    w = _c(w_i8, np.int8)
    assert w.size % 4 == 0
    out = np.empty((w.size // 4,), np.uint8)
    bad = lib().orc_pack_ref(_p(w, ctypes.c_int8), ctypes.c_long(w.size), _p(out, ctypes.c_uint8))
    return out, int(bad)


def unpack_ref(packed_u8, shape):
    p = _c(packed_u8, np.uint8)
    out = np.empty((p.size * 4,), np.int8)
    lib().orc_unpack_ref(_p(p, ctypes.c_uint8), ctypes.c_long(out.size), _p(out, ctypes.c_int8))
    return out.reshape(shape)
