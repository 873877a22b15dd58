"""CPU fp64 oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2606_16317_b200/ and shares no code with it.
"""
from .oracle import (  # noqa: F401
    MODE_DENSE,
    MODE_DYNAMIC,
    MODE_FIXED,
    OracleResult,
    build,
    dense_attention_textbook,
    lambda_from_preal,
    lambda_from_recall,
    max_threads,
    run_head,
)
from .brute_force import brute_force_head  # noqa: F401
from .reorder import brick_permutation, reorder  # noqa: F401
from .block_mass import block_mass, block_sqmass, eq3_lhs, select_greedy, select_topk, select_topp  # noqa: F401
from .analysis import KURTOSIS_BINS, excess_kurtosis, kurtosis_bin, row_probabilities, row_topk_curve, table3  # noqa: F401
