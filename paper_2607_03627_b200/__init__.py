"""B200-native restarted PDHG LP solver for DC unit-commitment LPs (arxiv/paper_2607_03627, GPU half).

Thin ctypes binding over the C ABI of include/uc_pdhg.h: argument marshalling only -- every step of
the method runs in the CUDA kernels of csrc/.  There is no CPU path: without the compiled extension
or without a GPU every compute call raises.
"""
from .binding import (UcLp, Options, Params, Result, Info, Solution, UcError, default_params, default_options,
                      load_library, library_path, solve_batch, release_scratch, STATUS_NAMES,
                      OPTIMAL, ITERATION_LIMIT, CANCELLED, TIME_LIMIT, NUMERICAL_ERROR,
                      ATTEMPT_DTYPE, CHECK_DTYPE)

__all__ = ["UcLp", "Options", "Params", "Result", "Info", "Solution", "UcError", "default_params", "default_options",
           "load_library", "library_path", "solve_batch", "release_scratch", "STATUS_NAMES", "OPTIMAL", "ITERATION_LIMIT", "CANCELLED", "TIME_LIMIT",
           "NUMERICAL_ERROR", "ATTEMPT_DTYPE", "CHECK_DTYPE"]
