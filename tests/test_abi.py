"""CPU-side tests of the C-ABI boundary: the library loads, exports every symbol the header declares,
validates its arguments on the host before touching a device, and has no CPU fallback."""
import ctypes
import math
import os
import re

import numpy as np
import pytest
import torch

import paper_2606_16317_b200 as sa
from paper_2606_16317_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "sparse_attn.h")


@pytest.fixture(scope="module", autouse=True)
def built():
    build.build()


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sparse_attn_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    declared = _declared_functions()
    assert "sparse_attn_fwd" in declared and len(declared) >= 8
    lib = ctypes.CDLL(sa.library_path())
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/sparse_attn.h but not exported"
    assert sorted(binding.EXPORTED_SYMBOLS) == declared
    assert sa.version() == 100


def test_params_struct_matches_header_layout():
    # uint32, float, float, int32, int32, (pad), void*, uint8_t*, float*, const uint8_t*, uint64_t*
    assert ctypes.sizeof(sa.SparseAttnParams) == 64
    assert sa.SparseAttnParams.stream.offset == 24
    assert sa.SparseAttnParams.skip_mask_in.offset == 48
    assert sa.SparseAttnParams.cycles_out.offset == 56


def test_lambda_helpers():
    assert abs(sa.lambda_from_recall(0.9, 1024) - math.log(0.1 / 1024)) < 1e-12
    assert abs(sa.lambda_from_preal(1.5, 128, 75600) - (math.log(1.5) + math.log(128 / 75600))) < 1e-12  # Eq. 7
    assert abs(sa.lambda_from_preal(1.5, 128, 75600) - (-6.0)) < 0.03


def _bufs(n=4096):
    a = np.zeros(n + 64, dtype=np.uint8)
    off = (-a.ctypes.data) % 64
    return a, a.ctypes.data + off


@pytest.mark.parametrize("case,status", [
    ("null_q", -1), ("null_out", -1), ("bad_B", -2), ("bad_N", -2), ("bad_D", -3), ("bad_tile", -4),
    ("bad_mode", -5), ("null_params_sparse", -6), ("nan_lambda", -6), ("positive_lambda_fixed", -6),
    ("bad_struct_size", -6), ("negative_scale", -6), ("misaligned", -7), ("too_many_heads", -2),
    ("mask_mode_without_mask", -6), ("mask_in_other_mode", -6), ("mask_mode_narrow_tile", -4),
])
def test_error_paths_checked_on_host(case, status):
    keep, ptr = _bufs()
    q = k = v = out = ptr
    B, H, N, D, mode = 1, 1, 16, 64, sa.MODE_DYNAMIC
    p = sa.make_params(lam=-2.0)
    if case == "null_q":
        q = None
    elif case == "null_out":
        out = None
    elif case == "bad_B":
        B = 0
    elif case == "bad_N":
        N = -5
    elif case == "bad_D":
        D = 96
    elif case == "bad_tile":
        p.tile_q = 32
    elif case == "bad_mode":
        mode = 4
    elif case == "null_params_sparse":
        p = None
    elif case == "nan_lambda":
        p.lambda_ = float("nan")
    elif case == "positive_lambda_fixed":
        p.lambda_, mode = 0.5, sa.MODE_FIXED
    elif case == "mask_mode_without_mask":
        mode = sa.MODE_MASK
    elif case == "mask_in_other_mode":
        p.skip_mask_in = 4096
    elif case == "mask_mode_narrow_tile":
        p.skip_mask_in, p.tile_q, p.tile_k, mode, D = 4096, 128, 32, sa.MODE_MASK, 128
    elif case == "bad_struct_size":
        p.struct_size = 12
    elif case == "negative_scale":
        p.softmax_scale = -1.0
    elif case == "misaligned":
        q = ptr + 2
    elif case == "too_many_heads":
        B, H = 300, 300
    with pytest.raises(sa.SparseAttnError) as e:
        sa.sparse_attn_fwd(q, k, v, out, None, B, H, N, D, p, mode, None)
    assert e.value.status == status
    assert sa.last_error() != ""
    assert sa.status_string(status) != "unknown status"
    del keep


def test_dense_mode_accepts_null_params_until_device_check():
    keep, ptr = _bufs()
    if torch.cuda.is_available():
        pytest.skip("device present: covered by the gpu tests")
    with pytest.raises(sa.SparseAttnError) as e:
        sa.sparse_attn_fwd(ptr, ptr, ptr, ptr, None, 1, 1, 16, 64, None, sa.MODE_DENSE, None)
    assert e.value.status == -8          # no CPU fallback: without an sm_100 device the call fails loudly
    with pytest.raises(sa.SparseAttnError) as e:
        sa.sparse_attn_fwd_host(ptr, ptr, ptr, ptr, None, 1, 1, 16, 64, None, sa.MODE_DENSE, None)
    assert e.value.status == -8
    del keep


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_16317_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle|dynsparse_oracle", text, flags=re.M), f

    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2606_16317_b200", text, flags=re.M)
