"""CPU-side checks of the boundary (no GPU): the C-ABI library loads and exports every symbol that
include/uc_pdhg.h and include/uc_pdhg_hooks.h declare, struct layouts match the header, argument validation answers before any
device is touched, and the product path fails loudly (never falls back) without a GPU."""
import ctypes as C
import math
import os
import re

import numpy as np
import pytest

import paper_2607_03627_b200 as P
from paper_2607_03627_b200 import binding
from workloads import tiny

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_functions():
    src = "".join(open(os.path.join(ROOT, "include", h)).read() for h in ("uc_pdhg.h", "uc_pdhg_hooks.h"))
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(uc_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    lib = P.load_library()
    names = header_functions()
    assert {"uc_lp_create", "uc_pdhg_solve", "uc_pdhg_cancel", "uc_lp_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert set(binding.EXPORTS) == set(names)
    # the product header carries no measurement or test hook; they live in uc_pdhg_hooks.h
    product = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "uc_pdhg.h")).read(), flags=re.S)
    for hook in ("uc_pdhg_time_kernels", "uc_pdhg_timeline", "uc_lp_compare_layout", "uc_host_layout_selftest", "uc_host_log_rounded"):
        assert hook not in product, hook


def test_default_structs_match_header_values():
    o = P.default_options()
    assert (o.device, o.ruiz_iters, o.pc_alpha, o.sell_window, o.long_row_threshold) == (-1, 10, 1.0, 4096, 32)
    p = P.default_params()
    # PAPER.md l.66 / l.91: iteration limit 100,000; convergence tolerance 1e-4
    assert p.iter_limit == 100000 and p.eps_rel == 1e-4 and p.eps_abs == 1e-4 and math.isinf(p.time_limit_s)
    assert (p.beta_sufficient, p.beta_necessary, p.beta_artificial, p.weight_smoothing) == (0.2, 0.8, 0.36, 0.5)
    assert p.check_every == 64 and p.fixed_iterations == 0 and not p.x0 and not p.stream


def test_struct_layouts_match_a_c_client_compiled_against_the_header(tmp_path):
    """A C11 client built with gcc against include/uc_pdhg.h prints sizeof and every offsetof; the ctypes Structures and the
    numpy record dtypes of the binding must give the same numbers (a reordered field of equal type would pass a
    default-value check, not this one)."""
    import shutil
    import subprocess
    structs = {"uc_lp_options": binding.Options, "uc_pdhg_params": binding.Params, "uc_pdhg_result": binding.Result,
               "uc_lp_info": binding.Info}
    records = {"uc_attempt_record": binding.ATTEMPT_DTYPE, "uc_check_record": binding.CHECK_DTYPE}
    lines = ["#include <stdio.h>", "#include <stddef.h>", '#include "uc_pdhg.h"', "int main(void) {"]
    for name, st in structs.items():
        lines.append(f'printf("{name} size %zu\\n", sizeof({name}));')
        lines += [f'printf("{name} {f} %zu\\n", offsetof({name}, {f}));' for f, _ in st._fields_]
    for name, dt in records.items():
        lines.append(f'printf("{name} size %zu\\n", sizeof({name}));')
        lines += [f'printf("{name} {f} %zu\\n", offsetof({name}, {f}));' for f in dt.names]
    lines += ['printf("UC_SPMV_STATIC_MAX_DOUBLES size %d\\n", (int)UC_SPMV_STATIC_MAX_DOUBLES);', "return 0; }"]
    src = tmp_path / "client.c"; exe = tmp_path / "client"
    src.write_text("\n".join(lines))
    gcc = shutil.which("gcc")
    assert gcc, "gcc is part of the image"
    subprocess.check_call([gcc, "-std=c11", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)])
    got = {}
    for ln in subprocess.check_output([str(exe)], text=True).splitlines():
        a, b, c = ln.split()
        got[(a, b)] = int(c)
    for name, st in structs.items():
        assert got[(name, "size")] == C.sizeof(st), name
        for f, _ in st._fields_:
            assert got[(name, f)] == getattr(st, f).offset, (name, f)
    for name, dt in records.items():
        assert got[(name, "size")] == dt.itemsize, name
        for f in dt.names:
            assert got[(name, f)] == dt.fields[f][1], (name, f)
    assert got[("UC_SPMV_STATIC_MAX_DOUBLES", "size")] == binding.SPMV_STATIC_MAX_DOUBLES
    # and the header declares exactly the fields the binding knows (a field added on one side only fails here)
    hdr = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "uc_pdhg.h")).read(), flags=re.S)
    for name, st in list(structs.items()) + [(k, None) for k in records]:
        body = re.search(r"typedef struct \{([^}]*)\} " + name + ";", hdr).group(1)
        declared = []
        for decl in body.split(";"):
            decl = decl.strip()
            if not decl:
                continue
            names = decl.split(None, 1)[1] if not decl.startswith("const") else decl.split(None, 2)[2]
            declared += [t.strip().lstrip("*").strip() for t in names.split(",")]
        want = [f for f, _ in st._fields_] if st is not None else list(records[name].names)
        assert declared == want, name


def _create_raw(lp, **over):
    lib = P.load_library()
    a = dict(row_ptr=lp.row_ptr, col_idx=lp.col_idx, val=lp.val, sense=lp.sense, b=lp.b, c=lp.c, l=lp.l, u=lp.u)
    a.update(over)
    keep = {k: (None if v is None else np.ascontiguousarray(v)) for k, v in a.items()}
    ptr = lambda v: None if v is None else C.c_void_p(v.ctypes.data)
    h = C.c_void_p()
    rc = lib.uc_lp_create(over.get("m", lp.m), over.get("n", lp.n), int(lp.row_ptr[-1]),
                          *[ptr(keep[k]) for k in ("row_ptr", "col_idx", "val", "sense", "b", "c", "l", "u")],
                          None, C.cast(C.byref(h), C.c_void_p))
    return rc, lib.uc_last_error().decode(), h


def test_invalid_arguments_are_rejected_before_touching_a_device():
    lp = tiny.small_random(6, 4, 0)
    rc, msg, _ = _create_raw(lp, col_idx=np.where(np.arange(lp.nnz) == 1, 99, lp.col_idx).astype(np.int32))
    assert rc == -1 and "column index" in msg
    dup = lp.col_idx.copy(); dup[1] = dup[0]
    assert lp.row_ptr[1] >= 2
    rc, msg, _ = _create_raw(lp, col_idx=dup)
    assert rc == -1 and "duplicate" in msg
    rc, msg, _ = _create_raw(lp, sense=np.full(lp.m, ord("L"), np.uint8))
    assert rc == -1 and "sense" in msg
    rc, msg, _ = _create_raw(lp, l=lp.u + 1.0)
    assert rc == -1 and "l > u" in msg
    bad = lp.val.copy(); bad[0] = np.nan
    rc, msg, _ = _create_raw(lp, val=bad)
    assert rc == -1 and "non-finite" in msg
    rc, msg, _ = _create_raw(lp, b=None)
    assert rc == -1
    lib = P.load_library()
    assert lib.uc_pdhg_cancel(None) == -1
    assert lib.uc_pdhg_solve(None, None, None, None, None) == -1
    lib.uc_lp_destroy(None)                                   # NULL is fine
    assert lib.uc_lp_update_objective(None, None) == -1 and lib.uc_lp_update_bounds(None, None, None) == -1
    res = (binding.Result * 2)()
    two_null = (C.c_void_p * 2)(None, None)
    assert lib.uc_pdhg_solve_batch(C.cast(two_null, C.c_void_p), 2, None, None, None, C.cast(res, C.c_void_p), 0) == -1
    assert lib.uc_pdhg_solve_batch(None, 0, None, None, None, None, 0) == 0      # an empty batch is not an error


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(P.UcError) as e:
        P.UcLp(tiny.two_var())
    assert e.value.code == -2 and "no CPU path" in str(e.value)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_03627_b200")
    for base, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                txt = open(os.path.join(base, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "pdhg_oracle" not in txt, f
    osrc = open(os.path.join(ROOT, "oracle", "pdhg_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "import paper_2607_03627_b200" not in osrc and "uc_pdhg.h" not in osrc and "csrc" not in osrc


def test_double_double_log_exp_are_correctly_rounded():
    """The primal-weight update (R11) uses exp/log; the device evaluates them in double-double
    (csrc/uc_dd.cuh).  Same source compiled for the host, against 200-bit mpmath."""
    mp = pytest.importorskip("mpmath")
    mp.mp.prec = 200
    lib = P.load_library()
    rng = np.random.default_rng(0)
    for a in np.concatenate([np.exp(rng.uniform(-40, 40, 3000)), [1.0, 2.0, 0.5, 1e-10, 1e10, 1.0000000000000002]]):
        assert lib.uc_host_log_rounded(float(a)) == float(mp.log(mp.mpf(float(a))))
    for x in np.concatenate([rng.uniform(-60, 60, 3000), [0.0, 1.0, -1.0, 1e-17]]):
        assert lib.uc_host_exp_rounded(float(x)) == float(mp.exp(mp.mpf(float(x))))
