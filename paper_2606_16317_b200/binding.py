"""ctypes binding of include/sparse_attn.h -- argument marshalling only.

`sparse_attn_fwd` takes torch CUDA tensors (torch is used for device memory and streams, nothing
else) or raw device pointers, and calls the C entry point of the same name.  The extension must
have been built (`python -m paper_2606_16317_b200.build` or `__graft_entry__.build()`); loading
fails loudly otherwise -- there is no fallback path.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

MODE_DENSE, MODE_FIXED, MODE_DYNAMIC, MODE_MASK = 0, 1, 2, 3
SELECT_TOPK, SELECT_TOPP = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("SPARSE_ATTN_LIB") or os.path.join(_HERE, "libsparse_attn.so")
_lib = None

# every symbol include/sparse_attn.h declares
EXPORTED_SYMBOLS = (
    "sparse_attn_fwd",
    "sparse_attn_fwd_host",
    "sparse_attn_release_scratch",
    "sparse_attn_lambda_from_recall",
    "sparse_attn_lambda_from_preal",
    "sparse_attn_block_mass",
    "sparse_attn_block_stats",
    "sparse_attn_select_blocks_greedy",
    "sparse_attn_recall_stats",
    "sparse_attn_output_error",
    "sparse_attn_row_topk_curve",
    "sparse_attn_row_topk_curve_static",
    "sparse_attn_brick_permutation",
    "sparse_attn_reorder_tokens",
    "sparse_attn_select_blocks",
    "sparse_attn_status_string",
    "sparse_attn_last_error",
    "sparse_attn_version",
    "sparse_attn_launch_count",
)


class SparseAttnError(RuntimeError):
    def __init__(self, status: int, detail: str):
        super().__init__(f"sparse_attn status {status} ({status_string(status)}): {detail}")
        self.status = status
        self.detail = detail


class SparseAttnParams(ctypes.Structure):
    """Mirror of `sparse_attn_params` (include/sparse_attn.h)."""
    _fields_ = [
        ("struct_size", ctypes.c_uint32),
        ("lambda_", ctypes.c_float),
        ("softmax_scale", ctypes.c_float),
        ("tile_q", ctypes.c_int32),
        ("tile_k", ctypes.c_int32),
        ("stream", ctypes.c_void_p),
        ("skip_mask_out", ctypes.c_void_p),
        ("margin_out", ctypes.c_void_p),
        ("skip_mask_in", ctypes.c_void_p),
        ("cycles_out", ctypes.c_void_p),
    ]


def library_path() -> str:
    return _LIB_PATH


def _load():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(
                f"{_LIB_PATH} is missing: build the CUDA extension first "
                "(python -m paper_2606_16317_b200.build). There is no CPU fallback.")
        lib = ctypes.CDLL(_LIB_PATH)
        fwd_args = [ctypes.c_void_p] * 5 + [ctypes.c_int] * 4 + [ctypes.POINTER(SparseAttnParams), ctypes.c_int,
                                                                 ctypes.c_void_p]
        lib.sparse_attn_fwd.restype = ctypes.c_int
        lib.sparse_attn_fwd.argtypes = fwd_args
        lib.sparse_attn_fwd_host.restype = ctypes.c_int
        lib.sparse_attn_fwd_host.argtypes = fwd_args
        lib.sparse_attn_release_scratch.restype = ctypes.c_int
        lib.sparse_attn_release_scratch.argtypes = []
        lib.sparse_attn_lambda_from_recall.restype = ctypes.c_double
        lib.sparse_attn_lambda_from_recall.argtypes = [ctypes.c_double, ctypes.c_int]
        lib.sparse_attn_lambda_from_preal.restype = ctypes.c_double
        lib.sparse_attn_lambda_from_preal.argtypes = [ctypes.c_double, ctypes.c_int, ctypes.c_int]
        lib.sparse_attn_block_mass.restype = ctypes.c_int
        lib.sparse_attn_block_mass.argtypes = [ctypes.c_void_p] * 4 + [ctypes.c_int] * 4 + [ctypes.c_float, ctypes.c_void_p]
        lib.sparse_attn_block_stats.restype = ctypes.c_int
        lib.sparse_attn_block_stats.argtypes = [ctypes.c_void_p] * 5 + [ctypes.c_int] * 4 + [ctypes.c_float, ctypes.c_void_p]
        lib.sparse_attn_select_blocks_greedy.restype = ctypes.c_int
        lib.sparse_attn_select_blocks_greedy.argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_int] * 5 + [ctypes.c_double, ctypes.c_void_p]
        lib.sparse_attn_recall_stats.restype = ctypes.c_int
        lib.sparse_attn_recall_stats.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
        lib.sparse_attn_output_error.restype = ctypes.c_int
        lib.sparse_attn_output_error.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
        lib.sparse_attn_row_topk_curve.restype = ctypes.c_int
        lib.sparse_attn_row_topk_curve.argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_int] * 4 + [ctypes.c_float, ctypes.c_void_p,
                                                   ctypes.c_int, ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 4
        lib.sparse_attn_row_topk_curve_static.restype = ctypes.c_int
        lib.sparse_attn_row_topk_curve_static.argtypes = lib.sparse_attn_row_topk_curve.argtypes
        lib.sparse_attn_select_blocks.restype = ctypes.c_int
        lib.sparse_attn_select_blocks.argtypes = [ctypes.c_void_p, ctypes.c_void_p] + [ctypes.c_int] * 5 + [
            ctypes.c_double, ctypes.c_void_p]
        lib.sparse_attn_brick_permutation.restype = ctypes.c_int
        lib.sparse_attn_brick_permutation.argtypes = [ctypes.c_int] * 6 + [ctypes.c_void_p]
        lib.sparse_attn_reorder_tokens.restype = ctypes.c_int
        lib.sparse_attn_reorder_tokens.argtypes = [ctypes.c_void_p, ctypes.c_void_p] + [ctypes.c_int] * 4 + [
            ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
        lib.sparse_attn_status_string.restype = ctypes.c_char_p
        lib.sparse_attn_status_string.argtypes = [ctypes.c_int]
        lib.sparse_attn_last_error.restype = ctypes.c_char_p
        lib.sparse_attn_last_error.argtypes = []
        lib.sparse_attn_version.restype = ctypes.c_int
        lib.sparse_attn_launch_count.restype = ctypes.c_int64
        _lib = lib
    return _lib


def version() -> int:
    return _load().sparse_attn_version()


def launch_count() -> int:
    return _load().sparse_attn_launch_count()


def status_string(status: int) -> str:
    return _load().sparse_attn_status_string(int(status)).decode()


def last_error() -> str:
    return _load().sparse_attn_last_error().decode()


def sparse_attn_release_scratch() -> int:
    """C entry point `sparse_attn_release_scratch`: hand the scratch `sparse_attn_fwd_host` retains on the current device
    back to the driver."""
    rc = _load().sparse_attn_release_scratch()
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


def lambda_from_recall(recall: float, N: int) -> float:
    return _load().sparse_attn_lambda_from_recall(float(recall), int(N))


def lambda_from_preal(p_real: float, tile_k: int, N: int) -> float:
    return _load().sparse_attn_lambda_from_preal(float(p_real), int(tile_k), int(N))


def _ptr(x) -> Optional[int]:
    """Device/host address of a torch tensor, numpy array, int or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(f"cannot take the address of {type(x)}")


def make_params(lam: float = float("-inf"), softmax_scale: float = 0.0, tile_q: int = 0, tile_k: int = 0,
                stream=None, skip_mask_out=None, margin_out=None, skip_mask_in=None, cycles_out=None) -> SparseAttnParams:
    p = SparseAttnParams()
    p.struct_size = ctypes.sizeof(SparseAttnParams)
    p.lambda_ = lam
    p.softmax_scale = softmax_scale
    p.tile_q = tile_q
    p.tile_k = tile_k
    p.stream = _ptr(stream)
    p.skip_mask_out = _ptr(skip_mask_out)
    p.margin_out = _ptr(margin_out)
    p.skip_mask_in = _ptr(skip_mask_in)
    p.cycles_out = _ptr(cycles_out)
    return p


def _call(fn, q, k, v, out, lse, B, H, N, D, params, mode, stats_out):
    rc = fn(_ptr(q), _ptr(k), _ptr(v), _ptr(out), _ptr(lse), int(B), int(H), int(N), int(D),
            ctypes.byref(params) if params is not None else None, int(mode), _ptr(stats_out))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


def sparse_attn_fwd(q, k, v, out, lse, B, H, N, D, threshold_params, mode, stats_out):
    """C entry point `sparse_attn_fwd` (device buffers).  Tensors or raw pointers; see the header.

    Enqueues on threshold_params.stream (torch's current stream if the caller passed it there) and
    returns; the caller synchronises.
    """
    return _call(_load().sparse_attn_fwd, q, k, v, out, lse, B, H, N, D, threshold_params, mode, stats_out)


def sparse_attn_fwd_host(q, k, v, out, lse, B, H, N, D, threshold_params, mode, stats_out):
    """C entry point `sparse_attn_fwd_host` (host buffers; copies inside, synchronous)."""
    return _call(_load().sparse_attn_fwd_host, q, k, v, out, lse, B, H, N, D, threshold_params, mode, stats_out)


def sparse_attn_brick_permutation(grid_t, grid_h, grid_w, brick_t, brick_h, brick_w, perm_out):
    """C entry point `sparse_attn_brick_permutation` (pure host function; perm_out: host int32 [N], numpy or address)."""
    rc = _load().sparse_attn_brick_permutation(int(grid_t), int(grid_h), int(grid_w), int(brick_t), int(brick_h),
                                               int(brick_w), _ptr(perm_out))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


def sparse_attn_reorder_tokens(src, dst, B, H, N, D, perm, inverse, stream=None):
    """C entry point `sparse_attn_reorder_tokens` (device buffers; perm: device int32 [N])."""
    rc = _load().sparse_attn_reorder_tokens(_ptr(src), _ptr(dst), int(B), int(H), int(N), int(D), _ptr(perm),
                                            int(inverse), _ptr(stream))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


def sparse_attn_block_mass(q, k, lse, mass_out, B, H, N, D, softmax_scale=0.0, stream=None):
    """C entry point `sparse_attn_block_mass` (device buffers): per-tile mass of the dense attention probabilities."""
    rc = _load().sparse_attn_block_mass(_ptr(q), _ptr(k), _ptr(lse), _ptr(mass_out), int(B), int(H), int(N), int(D),
                                        float(softmax_scale), _ptr(stream))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


def sparse_attn_block_stats(q, k, lse, mass_out, sqmass_out, B, H, N, D, softmax_scale=0.0, stream=None):
    """C entry point `sparse_attn_block_stats` (device buffers): per-tile sums of p and of p^2 of the dense probabilities."""
    rc = _load().sparse_attn_block_stats(_ptr(q), _ptr(k), _ptr(lse), _ptr(mass_out), _ptr(sqmass_out), int(B), int(H), int(N),
                                         int(D), float(softmax_scale), _ptr(stream))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


def sparse_attn_select_blocks_greedy(mass, sqmass, skip_mask_out, B, H, N, tile_q, T_c, theta, stream=None):
    """C entry point `sparse_attn_select_blocks_greedy` (device buffers): the section-3 mask under Eq. 3's bound."""
    rc = _load().sparse_attn_select_blocks_greedy(_ptr(mass), _ptr(sqmass), _ptr(skip_mask_out), int(B), int(H), int(N),
                                                  int(tile_q), int(T_c), float(theta), _ptr(stream))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


def sparse_attn_recall_stats(lse_retained, lse_dense, n_rows, stats_out, stream=None):
    """C entry point `sparse_attn_recall_stats`: stats_out (device double[2]) = {min, sum} of e^(lse_retained - lse_dense)."""
    rc = _load().sparse_attn_recall_stats(_ptr(lse_retained), _ptr(lse_dense), int(n_rows), _ptr(stats_out), _ptr(stream))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


def sparse_attn_output_error(out_a, out_b, n_elems, stats_out, stream=None):
    """C entry point `sparse_attn_output_error`: stats_out (device double[2]) = {max, sum} of |a - b| over bf16 elements."""
    rc = _load().sparse_attn_output_error(_ptr(out_a), _ptr(out_b), int(n_elems), _ptr(stats_out), _ptr(stream))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


def sparse_attn_select_blocks(mass, skip_mask_out, B, H, T_r, T_c, kind, param, stream=None):
    """C entry point `sparse_attn_select_blocks` (device buffers): Top-K / Top-P bitmap from a block-mass matrix."""
    rc = _load().sparse_attn_select_blocks(_ptr(mass), _ptr(skip_mask_out), int(B), int(H), int(T_r), int(T_c), int(kind),
                                           float(param), _ptr(stream))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


def sparse_attn_row_topk_curve(q, k, v, B, H, N, D, rows, keep_counts, kurtosis_out, recall_out, mae_out, softmax_scale=0.0,
                               stream=None):
    """C entry point `sparse_attn_row_topk_curve` (Appendix A.1): rows = host int32 [n_rows, 2] (numpy), keep_counts = host
    int32 [n_keep] (numpy); q, k, v and the three fp64 outputs are device buffers."""
    n_rows, n_keep = int(rows.shape[0]), int(keep_counts.shape[0])
    rc = _load().sparse_attn_row_topk_curve(_ptr(q), _ptr(k), _ptr(v), int(B), int(H), int(N), int(D), float(softmax_scale),
                                            _ptr(rows), n_rows, _ptr(keep_counts), n_keep, _ptr(kurtosis_out),
                                            _ptr(recall_out), _ptr(mae_out), _ptr(stream))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc


# limits of the allocation-free entry point (include/sparse_attn.h: SPARSE_ATTN_STATIC_*)
STATIC_SCRATCH_FLOATS, STATIC_MAX_ROWS, STATIC_MAX_KEEP = 4 << 20, 2048, 4096


def sparse_attn_row_topk_curve_static(q, k, v, B, H, N, D, rows, keep_counts, kurtosis_out, recall_out, mae_out,
                                      softmax_scale=0.0, stream=None):
    """C entry point `sparse_attn_row_topk_curve_static`: the Appendix A.1 row curve for hosts that cannot allocate device
    memory -- a process whose HBM has all been handed to another allocator (any cudaMalloc would fail), or a request path
    that must not call the driver's allocator.  Same arguments and results as `sparse_attn_row_topk_curve`; the kernel's
    working memory is a fixed 16 MiB array inside the library, so n_rows * N <= STATIC_SCRATCH_FLOATS, n_rows <=
    STATIC_MAX_ROWS, n_keep <= STATIC_MAX_KEEP (SparseAttnError with status -2 beyond).  Every call on a device shares that
    one array: calls that may overlap on the GPU race.  The first call on a device looks the array's address up; make it
    before any stream capture."""
    n_rows, n_keep = int(rows.shape[0]), int(keep_counts.shape[0])
    rc = _load().sparse_attn_row_topk_curve_static(_ptr(q), _ptr(k), _ptr(v), int(B), int(H), int(N), int(D),
                                                   float(softmax_scale), _ptr(rows), n_rows, _ptr(keep_counts), n_keep,
                                                   _ptr(kurtosis_out), _ptr(recall_out), _ptr(mae_out), _ptr(stream))
    if rc != 0:
        raise SparseAttnError(rc, last_error())
    return rc
