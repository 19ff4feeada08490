"""Thin ctypes binding of libvlaternary.so (include/vla_ternary.h) -- argument marshalling only.

Every function has the name and argument order of its C entry point, takes torch CUDA tensors (or
raw integer device pointers) for the device buffers, passes `tensor.data_ptr()` and the current
torch CUDA stream, and raises VlaError on a non-zero vla_status.  Nothing is computed here: every
step of Eq. 4 runs in the library's kernels.  There is no fallback: if the
shared library cannot be loaded the import of this module fails.
"""
import ctypes
import os

import torch

from . import build as _build

VLA_OK = 0
(VLA_ERR_NULL, VLA_ERR_SHAPE, VLA_ERR_ALIGN, VLA_ERR_VALUE, VLA_ERR_DTYPE, VLA_ERR_WORKSPACE,
 VLA_ERR_ARCH, VLA_ERR_CUDA) = range(1, 9)
VLA_F32, VLA_BF16, VLA_I32 = 0, 1, 2
VLA_PATH_AUTO, VLA_PATH_SMALL_ALU, VLA_PATH_SMALL_TC, VLA_PATH_LARGE = 0, 1, 2, 3

_TORCH_DTYPE = {VLA_F32: torch.float32, VLA_BF16: torch.bfloat16, VLA_I32: torch.int32}

EXPORTS = [
    "vla_ternary_packed_bytes", "vla_ternary_workspace_bytes", "vla_ternary_pack", "vla_ternary_unpack",
    "vla_act_quant", "vla_ternary_gemm", "vla_ternary_linear", "vla_ternary_linear_host",
    "vla_ternary_host_workspace_bytes", "vla_ternary_linear_static",
    "vla_ternary_auto_path", "vla_i8_mma_issue_probe", "vla_status_string", "vla_launch_count",
    "vla_cached_attention", "vla_cached_attention_workspace_bytes",
    "vla_ternary_gemm_grouped", "vla_program_bytes", "vla_program_build", "vla_program_run", "vla_program_run_host", "vla_program_run_host_async", "vla_program_release",
]


class vla_copy(ctypes.Structure):
    _fields_ = [("host", ctypes.c_void_p), ("dev", ctypes.c_void_p), ("bytes", ctypes.c_size_t)]


class vla_prog_linear(ctypes.Structure):
    _fields_ = [("packed", ctypes.c_void_p), ("w_scale", ctypes.c_void_p), ("out", ctypes.c_void_p),
                ("N", ctypes.c_int), ("out_dtype", ctypes.c_int)]


class vla_prog_stage(ctypes.Structure):
    _fields_ = [("x_bf16", ctypes.c_void_p), ("M", ctypes.c_int), ("K", ctypes.c_int), ("depends", ctypes.c_int),
                ("n_linears", ctypes.c_int), ("linears", ctypes.POINTER(vla_prog_linear)),
                ("xq_opt", ctypes.c_void_p), ("x_scale_opt", ctypes.c_void_p)]


class VlaError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        super().__init__("%s: %s" % (where, vla_status_string(status)))


def _load():
    so = _build.SO
    if not _build.is_current():
        _build.build()          # missing, or built from other sources (a stale binary must never be loaded silently);
                                # needs nvcc and raises if the toolchain is missing -- no fallback
    lib = ctypes.CDLL(so)
    vp, i, sz, st = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t, ctypes.c_int
    lib.vla_ternary_packed_bytes.restype = sz
    lib.vla_ternary_packed_bytes.argtypes = [i, i]
    lib.vla_ternary_workspace_bytes.restype = sz
    lib.vla_ternary_workspace_bytes.argtypes = [i, i, i, i]
    lib.vla_ternary_pack.restype = st
    lib.vla_ternary_pack.argtypes = [vp, i, i, vp, sz, vp]
    lib.vla_ternary_unpack.restype = st
    lib.vla_ternary_unpack.argtypes = [vp, i, i, vp, vp]
    lib.vla_act_quant.restype = st
    lib.vla_act_quant.argtypes = [vp, i, i, vp, vp, vp]
    lib.vla_ternary_gemm.restype = st
    lib.vla_ternary_gemm.argtypes = [vp, vp, vp, vp, i, i, i, vp, i, i, vp, sz, vp]
    lib.vla_ternary_linear.restype = st
    lib.vla_ternary_linear.argtypes = [vp, vp, vp, i, i, i, vp, i, i, vp, vp, vp, sz, vp]
    lib.vla_ternary_linear_static.restype = st
    lib.vla_ternary_linear_static.argtypes = [vp, vp, vp, i, i, i, vp, i, i, vp]
    lib.vla_ternary_linear_host.restype = st
    lib.vla_ternary_linear_host.argtypes = [vp, vp, vp, i, i, i, vp, i, i, vp, sz, vp]
    lib.vla_ternary_host_workspace_bytes.restype = sz
    lib.vla_ternary_host_workspace_bytes.argtypes = [i, i, i, i, i]
    lib.vla_ternary_auto_path.restype = i
    lib.vla_ternary_auto_path.argtypes = [i, i, i]
    lib.vla_i8_mma_issue_probe.restype = st
    lib.vla_i8_mma_issue_probe.argtypes = [i, i, ctypes.POINTER(ctypes.c_float)]
    lib.vla_status_string.restype = ctypes.c_char_p
    lib.vla_status_string.argtypes = [st]
    lib.vla_launch_count.restype = ctypes.c_ulonglong
    lib.vla_launch_count.argtypes = []
    ps = ctypes.POINTER(vla_prog_stage)
    lib.vla_program_bytes.restype = sz
    lib.vla_program_bytes.argtypes = [ps, i]
    lib.vla_program_build.restype = st
    lib.vla_program_build.argtypes = [ps, i, vp, sz, vp]
    lib.vla_program_run.restype = st
    lib.vla_program_run.argtypes = [vp, vp]
    lib.vla_ternary_gemm_grouped.restype = st
    lib.vla_ternary_gemm_grouped.argtypes = [ctypes.POINTER(vla_prog_linear), i, vp, vp, i, i, i, vp]
    lib.vla_program_run_host.restype = st
    lib.vla_program_run_host.argtypes = [vp, ctypes.POINTER(vla_copy), i, ctypes.POINTER(vla_copy), i, vp]
    lib.vla_program_run_host_async.restype = st
    lib.vla_program_run_host_async.argtypes = [vp, ctypes.POINTER(vla_copy), i, ctypes.POINTER(vla_copy), i, vp]
    lib.vla_program_release.restype = st
    lib.vla_program_release.argtypes = [vp]
    lib.vla_cached_attention_workspace_bytes.restype = sz
    lib.vla_cached_attention_workspace_bytes.argtypes = [i, i, i, i, i]
    lib.vla_cached_attention.restype = st
    lib.vla_cached_attention.argtypes = [vp, vp, vp, vp, i, i, i, i, i, vp, i, vp, sz, vp]
    return lib


_lib = _load()
LIB_PATH = _build.SO


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _check(status, where):
    if status != VLA_OK:
        raise VlaError(status, where)


def vla_status_string(status):
    return _lib.vla_status_string(int(status)).decode()


def vla_ternary_packed_bytes(N, K):
    return int(_lib.vla_ternary_packed_bytes(N, K))


def vla_ternary_workspace_bytes(M, N, K, path=VLA_PATH_AUTO):
    return int(_lib.vla_ternary_workspace_bytes(M, N, K, path))


def vla_ternary_auto_path(M, N, K):
    return int(_lib.vla_ternary_auto_path(M, N, K))


def vla_launch_count():
    """Number of kernels this library has launched in this process (for bench.py's gpu_launches)."""
    return int(_lib.vla_launch_count())


def vla_ternary_pack(w, N, K, packed, packed_bytes=None, stream=None):
    if packed_bytes is None:
        packed_bytes = packed.numel() * packed.element_size()
    _check(_lib.vla_ternary_pack(_ptr(w), N, K, _ptr(packed), packed_bytes, _stream(stream)), "vla_ternary_pack")


def vla_ternary_unpack(packed, N, K, w, stream=None):
    _check(_lib.vla_ternary_unpack(_ptr(packed), N, K, _ptr(w), _stream(stream)), "vla_ternary_unpack")


def vla_act_quant(x_bf16, M, K, xq, x_scale, stream=None):
    _check(_lib.vla_act_quant(_ptr(x_bf16), M, K, _ptr(xq), _ptr(x_scale), _stream(stream)), "vla_act_quant")


def vla_ternary_gemm(packed, w_scale, xq, x_scale, M, N, K, out, out_dtype, path=VLA_PATH_AUTO,
                     workspace=None, workspace_bytes=0, stream=None):
    _check(_lib.vla_ternary_gemm(_ptr(packed), _ptr(w_scale), _ptr(xq), _ptr(x_scale), M, N, K, _ptr(out),
                                 out_dtype, path, _ptr(workspace), workspace_bytes, _stream(stream)),
           "vla_ternary_gemm")


def vla_ternary_linear(packed, w_scale, x_bf16, M, N, K, out, out_dtype, path=VLA_PATH_AUTO,
                       xq_opt=None, x_scale_opt=None, workspace=None, workspace_bytes=0, stream=None):
    _check(_lib.vla_ternary_linear(_ptr(packed), _ptr(w_scale), _ptr(x_bf16), M, N, K, _ptr(out), out_dtype, path,
                                   _ptr(xq_opt), _ptr(x_scale_opt), _ptr(workspace), workspace_bytes,
                                   _stream(stream)), "vla_ternary_linear")


VLA_STATIC_MAX_MK, VLA_STATIC_MAX_M = 8388608, 16384


def vla_ternary_linear_static(packed, w_scale, x_bf16, M, N, K, out, out_dtype, path=VLA_PATH_AUTO, stream=None):
    """vla_ternary_linear with its scratch in a fixed array inside the library: allocates nothing (include/vla_ternary.h)."""
    _check(_lib.vla_ternary_linear_static(_ptr(packed), _ptr(w_scale), _ptr(x_bf16), M, N, K, _ptr(out), out_dtype, path,
                                          _stream(stream)), "vla_ternary_linear_static")


def vla_ternary_host_workspace_bytes(M, N, K, out_dtype, path=VLA_PATH_AUTO):
    return int(_lib.vla_ternary_host_workspace_bytes(M, N, K, out_dtype, path))


def vla_ternary_linear_host(packed, w_scale, x_bf16_host, M, N, K, out_host, out_dtype, path,
                            workspace, workspace_bytes, stream=None):
    """x_bf16_host / out_host: HOST tensors (pinned for asynchronous copies).  Synchronises the stream."""
    _check(_lib.vla_ternary_linear_host(_ptr(packed), _ptr(w_scale), _ptr(x_bf16_host), M, N, K, _ptr(out_host),
                                        out_dtype, path, _ptr(workspace), workspace_bytes, _stream(stream)),
           "vla_ternary_linear_host")


def vla_i8_mma_issue_probe(ctas, mmas_per_cta):
    ms = ctypes.c_float(0.0)
    _check(_lib.vla_i8_mma_issue_probe(ctas, mmas_per_cta, ctypes.byref(ms)), "vla_i8_mma_issue_probe")
    return float(ms.value)


def _marshal_stages(stages):
    """stages: list of dicts {x, M, K, depends, linears: [{packed, w_scale, out, N, out_dtype}], xq_opt, x_scale_opt}
    -> (ctypes array of vla_prog_stage, keep-alive list)."""
    arr = (vla_prog_stage * len(stages))()
    keep = []
    for si, sd in enumerate(stages):
        lins = (vla_prog_linear * len(sd["linears"]))()
        for li, ld in enumerate(sd["linears"]):
            lins[li] = vla_prog_linear(_ptr(ld["packed"]), _ptr(ld["w_scale"]), _ptr(ld["out"]), int(ld["N"]),
                                       int(ld["out_dtype"]))
        keep.append(lins)
        arr[si] = vla_prog_stage(_ptr(sd["x"]), int(sd["M"]), int(sd["K"]), int(sd.get("depends", 0)), len(lins), lins,
                                 _ptr(sd.get("xq_opt")), _ptr(sd.get("x_scale_opt")))
    return arr, keep


def make_linears(linears):
    """[{packed, w_scale, out, N, out_dtype}] -> ctypes array of vla_prog_linear (marshalled once, reusable)."""
    arr = (vla_prog_linear * len(linears))()
    for li, ld in enumerate(linears):
        arr[li] = vla_prog_linear(_ptr(ld["packed"]), _ptr(ld["w_scale"]), _ptr(ld["out"]), int(ld["N"]), int(ld["out_dtype"]))
    return arr


def vla_ternary_gemm_grouped(linears, xq, x_scale, M, K, path=VLA_PATH_AUTO, stream=None):
    """linears: a ctypes array from make_linears (or a list of dicts, marshalled on the fly)."""
    arr = linears if not isinstance(linears, (list, tuple)) else make_linears(linears)
    _check(_lib.vla_ternary_gemm_grouped(arr, len(arr), _ptr(xq), _ptr(x_scale), M, K, path, _stream(stream)),
           "vla_ternary_gemm_grouped")


def vla_program_bytes(stages):
    arr, _keep = _marshal_stages(stages)
    return int(_lib.vla_program_bytes(arr, len(stages)))


def vla_program_build(stages, prog_dev, prog_bytes=None, stream=None):
    arr, _keep = _marshal_stages(stages)
    if prog_bytes is None:
        prog_bytes = prog_dev.numel() * prog_dev.element_size()
    _check(_lib.vla_program_build(arr, len(stages), _ptr(prog_dev), prog_bytes, _stream(stream)), "vla_program_build")


def vla_program_run(prog_dev, stream=None):
    _check(_lib.vla_program_run(_ptr(prog_dev), _stream(stream)), "vla_program_run")


def make_copies(pairs):
    """[(host tensor, device tensor)] -> ctypes array of vla_copy (marshalled once, reusable across calls)."""
    arr = (vla_copy * len(pairs))()
    for k, (h, d) in enumerate(pairs):
        arr[k] = vla_copy(_ptr(h), _ptr(d), h.numel() * h.element_size())
    return arr


def vla_program_run_host(prog_dev, copies_in, copies_out, stream=None):
    """copies_in / copies_out: ctypes arrays from make_copies.  Synchronises the stream."""
    _check(_lib.vla_program_run_host(_ptr(prog_dev), copies_in, len(copies_in), copies_out, len(copies_out),
                                     _stream(stream)), "vla_program_run_host")


def vla_program_run_host_async(prog_dev, copies_in, copies_out, stream=None):
    """vla_program_run_host without the final synchronisation (the caller synchronises the stream or an event on it)."""
    _check(_lib.vla_program_run_host_async(_ptr(prog_dev), copies_in, len(copies_in), copies_out, len(copies_out),
                                           _stream(stream)), "vla_program_run_host_async")


def vla_cached_attention_workspace_bytes(Mq, Mc, n_q_heads, n_kv_heads, d_k):
    return int(_lib.vla_cached_attention_workspace_bytes(Mq, Mc, n_q_heads, n_kv_heads, d_k))


def vla_cached_attention(q_bf16, kc_bf16, vc_bf16, visible_opt, Mq, Mc, n_q_heads, n_kv_heads, d_k, out, out_dtype,
                         workspace=None, workspace_bytes=0, stream=None):
    _check(_lib.vla_cached_attention(_ptr(q_bf16), _ptr(kc_bf16), _ptr(vc_bf16), _ptr(visible_opt), Mq, Mc, n_q_heads,
                                     n_kv_heads, d_k, _ptr(out), out_dtype, _ptr(workspace), workspace_bytes,
                                     _stream(stream)), "vla_cached_attention")


def vla_program_release(prog_dev):
    _check(_lib.vla_program_release(_ptr(prog_dev)), "vla_program_release")


# ------------------------------------------------------------------ conveniences (allocation only)
def compile_program(stages, device="cuda"):
    """Allocates the device buffer of a program and compiles `stages` into it; returns the buffer (a uint8 tensor
    that must be kept alive, together with every tensor the stages point to, while the program is run)."""
    nbytes = vla_program_bytes(stages)
    if nbytes == 0:
        raise VlaError(VLA_ERR_SHAPE, "compile_program")
    buf = torch.zeros(nbytes + 256, dtype=torch.uint8, device=device)
    off = (-buf.data_ptr()) % 256
    prog = buf[off:off + nbytes]
    vla_program_build(stages, prog, nbytes)
    prog._vla_keep = buf
    return prog


def pack_weights(w_i8):
    """int8 [N,K] CUDA tensor -> uint8 packed tensor of vla_ternary_packed_bytes(N,K) bytes."""
    N, K = w_i8.shape
    nbytes = vla_ternary_packed_bytes(N, K)
    if nbytes == 0:
        raise VlaError(VLA_ERR_SHAPE, "pack_weights")
    packed = torch.empty(nbytes, dtype=torch.uint8, device=w_i8.device)
    vla_ternary_pack(w_i8.contiguous(), N, K, packed, nbytes)
    return packed


def empty_out(M, N, out_dtype, device="cuda"):
    return torch.empty((M, N), dtype=_TORCH_DTYPE[out_dtype], device=device)
