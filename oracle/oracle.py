"""ctypes front-end of oracle/dynsparse_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Builds the C oracle with gcc (OpenMP) next to its source and calls it.  The arithmetic of the
method lives in the C file; this module only marshals arrays and derives reports from the
oracle's own outputs.  `dense_attention_textbook` is the plain definition softmax(scale*QK^T)V
written with numpy, used to pin the C code's dense mode (P1).
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

MODE_DENSE, MODE_FIXED, MODE_DYNAMIC = 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dynsparse_oracle.c")
_LIB = os.path.join(_HERE, "libdynsparse_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.dynsparse_oracle_head.restype = ctypes.c_int
        lib.dynsparse_oracle_head.argtypes = [
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
            ctypes.c_double, ctypes.c_double, ctypes.c_int,
            ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
        lib.dynsparse_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    """Threads the oracle will actually use (OpenMP default, bounded by the affinity mask)."""
    n = _load().dynsparse_oracle_max_threads()
    try:
        n = min(n, len(os.sched_getaffinity(0)))
    except AttributeError:
        pass
    return max(1, n)


def lambda_from_recall(recall: float, N: int) -> float:
    """Worst-case threshold lambda = ln(eps / L) with eps = 1 - recall."""
    return math.log((1.0 - recall) / N)


def lambda_from_preal(p_real: float, tile_k: int, N: int) -> float:
    """Eq. 7: lambda = ln(P_real) + ln(B_c / L)."""
    return math.log(p_real) + math.log(tile_k / N)


@dataclass
class OracleResult:
    out: np.ndarray      # [n_qtiles, tile_q, D] fp64 (rows beyond N zero)
    lse: np.ndarray      # [n_qtiles, tile_q] fp64
    skip: np.ndarray     # [n_qtiles, T_c] uint8, 1 = skipped
    margin: np.ndarray   # [n_qtiles, T_c] fp64, g_ij = max_r t_r - lambda
    qtiles: np.ndarray   # [n_qtiles] int32
    N: int
    tile_q: int
    tile_k: int

    @property
    def skipped(self) -> int:
        return int(self.skip.sum())

    @property
    def executed(self) -> int:
        return int(self.skip.size - self.skip.sum())

    @property
    def sparsity(self) -> float:
        return self.skipped / self.skip.size

    def rows(self):
        """(out, lse) flattened to the valid rows, in (qtile, row) order."""
        outs, lses = [], []
        for t, i in enumerate(self.qtiles):
            rows = min(self.tile_q, self.N - int(i) * self.tile_q)
            outs.append(self.out[t, :rows])
            lses.append(self.lse[t, :rows])
        return np.concatenate(outs), np.concatenate(lses)


def run_head(q_bits: np.ndarray, k_bits: np.ndarray, v_bits: np.ndarray, *, tile: int, lam: float,
             mode: int, scale: Optional[float] = None, qtiles: Optional[Sequence[int]] = None,
             forced_skip: Optional[np.ndarray] = None, tile_k: Optional[int] = None,
             n_threads: int = 0) -> OracleResult:
    """Run the oracle on one head.  q/k/v: uint16 bf16 bit patterns [N, D]."""
    lib = _load()
    q_bits = np.ascontiguousarray(q_bits, dtype=np.uint16)
    k_bits = np.ascontiguousarray(k_bits, dtype=np.uint16)
    v_bits = np.ascontiguousarray(v_bits, dtype=np.uint16)
    N, D = q_bits.shape
    tile_q = tile
    tile_k = tile if tile_k is None else tile_k
    T_r, T_c = -(-N // tile_q), -(-N // tile_k)
    if scale is None:
        scale = 1.0 / math.sqrt(D)      # DESIGN.md G1
    qt = np.arange(T_r, dtype=np.int32) if qtiles is None else np.asarray(list(qtiles), dtype=np.int32)
    n = len(qt)
    out = np.zeros((n, tile_q, D), dtype=np.float64)
    lse = np.zeros((n, tile_q), dtype=np.float64)
    skip = np.zeros((n, T_c), dtype=np.uint8)
    margin = np.zeros((n, T_c), dtype=np.float64)
    forced_p = None
    if forced_skip is not None:
        forced_skip = np.ascontiguousarray(forced_skip, dtype=np.uint8)
        assert forced_skip.shape == (n, T_c)
        forced_p = forced_skip.ctypes.data
    rc = lib.dynsparse_oracle_head(
        q_bits.ctypes.data, k_bits.ctypes.data, v_bits.ctypes.data, N, D, tile_q, tile_k,
        float(scale), float(lam), int(mode), qt.ctypes.data, n, forced_p,
        out.ctypes.data, lse.ctypes.data, skip.ctypes.data, margin.ctypes.data, int(n_threads))
    if rc != 0:
        raise ValueError(f"dynsparse_oracle_head failed with {rc}")
    return OracleResult(out, lse, skip, margin, qt, N, tile_q, tile_k)


def dense_attention_textbook(q: np.ndarray, k: np.ndarray, v: np.ndarray, scale: float):
    """softmax(scale * Q K^T) V by the direct max-subtracted two-pass formula.

    q, k, v: float64 [N, D].  Returns (O [N, D], lse [N], P [N, N]).
    """
    s = scale * (q @ k.T)
    m = s.max(axis=1, keepdims=True)
    e = np.exp(s - m)
    z = e.sum(axis=1, keepdims=True)
    p = e / z
    return p @ v, (m + np.log(z))[:, 0], p
