"""C-ABI library checks that need no GPU: libbq.so builds, loads and exports every symbol include/*.h declares;
argument validation that happens before any device work; no silent CPU fallback."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bq():
    from paper_2111_04457_b200 import build
    build.build()
    from paper_2111_04457_b200 import bq as _bq
    return _bq


HEADERS = ("bq.h", "bq_test.h")     # the product boundary, and the test / benchmark hooks


def declared_symbols(headers=HEADERS):
    names = set()
    for hname in headers:
        with open(os.path.join(ROOT, "include", hname)) as f:
            text = re.sub(r"/\*.*?\*/", "", f.read(), flags=re.S)
        names |= set(re.findall(r"\b(bq_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_product_header_holds_only_the_boundary():
    """include/bq.h is SURVEY §8(b)'s boundary; the bq_blas_* / bq_bench_* / counter hooks live in bq_test.h."""
    prod = declared_symbols(("bq.h",))
    assert not [n for n in prod if n.startswith(("bq_blas_", "bq_bench_")) or n in ("bq_get_counters", "bq_schur_apply_dots")]
    for n in ("bq_lattice_create", "bq_gauge_load", "bq_wilson_apply", "bq_clover_apply", "bq_solve"):
        assert n in prod


def test_every_declared_symbol_is_exported(bq):
    lib = bq.lib()
    names = declared_symbols()
    assert set(names) == set(bq.EXPORTS), "binding and header disagree"
    for n in names:
        assert hasattr(lib, n), f"libbq.so does not export {n}"


def test_struct_layouts_match_header(bq):
    assert ctypes.sizeof(bq.bq_solve_opts) == 56
    assert ctypes.sizeof(bq.bq_solve_info) == 72


def test_status_strings(bq):
    lib = bq.lib()
    seen = {lib.bq_status_string(s).decode() for s in range(10)}
    assert len(seen) == 10 and "unknown status" not in seen


def test_extent_and_phase_validation_precede_device_work(bq):
    for L in ((3, 4, 4, 4), (4, 4, 4, 5), (0, 4, 4, 4), (4, 1, 4, 4)):
        with pytest.raises(bq.BqError) as e:
            bq.bq_lattice_create(*L)
        assert e.value.status == bq.BQ_EODD_EXTENT
    with pytest.raises(bq.BqError) as e:
        bq.bq_lattice_create(4, 4, 4, 4, [1, 1, 1, 0.5])       # |phase| != 1
    assert e.value.status == bq.BQ_EINVAL
    with pytest.raises(bq.BqError) as e:
        bq.bq_lattice_create(2048, 2048, 1024, 2)               # V >= 2^31
    assert e.value.status == bq.BQ_EINVAL


def test_no_cpu_fallback(bq):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    with pytest.raises(bq.BqError) as e:
        bq.bq_lattice_create(4, 4, 4, 4)
    assert e.value.status == bq.BQ_ECUDA


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2111_04457_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".c")):
                with open(os.path.join(dirpath, f)) as fh:
                    src = fh.read()
                assert "oracle" not in src.replace("the oracle", "").replace("oracle/", "").replace("CPU oracle", "").replace(
                    "oracle's", ""), f"{f} mentions the oracle module"


def test_header_is_plain_c_and_links(bq, tmp_path):
    """include/bq.h must be usable from plain C (the boundary is a C ABI): a C99 translation unit that includes it, takes
    the address of every declared function and fills the option / info structs compiles with gcc and links against libbq.so."""
    import subprocess
    names = declared_symbols()
    src = tmp_path / "abi_check.c"
    lines = ['#include "bq.h"', '#include "bq_test.h"', "#include <stddef.h>", "typedef void (*fn_t)(void);", "int main(void) {", "    fn_t fns[] = {"]
    lines += [f"        (fn_t){n}," for n in names]
    lines += ["    };", "    bq_solve_opts o = {0};", "    bq_solve_info info;", "    o.inner_prec = BQ_HALF; o.method = BQ_CGNR; o.lexical = 0; o.x0_zero = 1;",
              "    info.phase_seconds[4] = 0.0; info.inner_iters = (int)BQ_MODE_DDAGD;",
              "    return (fns[0] != NULL && o.x0_zero && info.inner_iters == 2) ? 0 : 1;", "}"]
    src.write_text("\n".join(lines) + "\n")
    libdir = os.path.join(ROOT, "paper_2111_04457_b200")
    exe = tmp_path / "abi_check"
    cmd = ["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe),
           "-L", libdir, "-l:libbq.so", f"-Wl,-rpath,{libdir}", "-Wl,--allow-shlib-undefined"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
