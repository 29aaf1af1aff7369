"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/rbg.h declares; the product path fails loudly without a GPU (no CPU fallback)."""
import re
from pathlib import Path

import pytest
import torch

ROOT = Path(__file__).resolve().parent.parent


def _declared():
    text = (ROOT / "include" / "rbg.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rbg_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2308_04869_b200.build import build
    build()
    import paper_2308_04869_b200 as rbg
    lib = rbg.load_library()
    declared = _declared()
    assert declared == rbg.exported_symbols()
    assert "rbg_create" in declared and "rbg_collision" in declared and "rbg_destroy" in declared
    for name in declared:
        assert getattr(lib, name) is not None


def test_header_is_plain_c():
    import subprocess
    src = '#include "rbg.h"\nint main(void){ rbg_spatial_grid g = {1,1,1,0}; (void)g; return 0; }\n'
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-fsyntax-only", "-I", str(ROOT / "include"), "-x", "c", "-"],
                   input=src.encode(), check=True)


def test_product_and_oracle_share_no_code():
    pat_oracle = re.compile(r"^\s*(import|from)\s+oracle\b|#include\s+[\"<][^\">]*oracle", re.M)
    for p in (ROOT / "paper_2308_04869_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            assert not pat_oracle.search(p.read_text()), p
    pat_prod = re.compile(r"^\s*(import|from)\s+paper_2308_04869_b200\b|#include\s+[\"<][^\">]*(rbg\.h|rbg_kernels)", re.M)
    for p in (ROOT / "oracle").rglob("*"):
        if p.suffix in (".py", ".cpp", ".h"):
            assert not pat_prod.search(p.read_text()), p
    for p in (ROOT / "workloads").rglob("*.py"):
        assert not pat_oracle.search(p.read_text()) and not pat_prod.search(p.read_text()), p


def _code_lines(path):
    """Source lines with comments and all white space removed; lines too short to say anything (braces, `break;`,
    `#pragma unroll`, `return 0;` ...) are dropped, so that a run is a run of statements."""
    text = path.read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    out = []
    for line in text.splitlines():
        line = re.sub(r"\s+", "", line.split("//", 1)[0])
        if len(line) >= 12 and not line.startswith("#"):
            out.append(line)
    return out


def test_no_block_of_oracle_source_repeats_in_the_product():
    """Parity compares the CUDA path with the oracle, so text that is the same on both sides is compared with itself
    (the role-expansion and deposit-factor blocks had been pasted).  No run of five or more consecutive
    statements may be identical between any oracle C++ file and any product source file."""
    RUN = 5
    oracle_files = [q for q in (ROOT / "oracle").rglob("*") if q.suffix in (".cpp", ".h", ".c")]
    product_files = [q for q in (ROOT / "paper_2308_04869_b200").rglob("*") if q.suffix in (".cu", ".cuh", ".h", ".cpp")]
    product_files.append(ROOT / "include" / "rbg.h")
    assert oracle_files and len(product_files) >= 4
    for po in oracle_files:
        lo = _code_lines(po)
        runs = {tuple(lo[i:i + RUN]): i for i in range(len(lo) - RUN + 1)}
        for pp in product_files:
            lp = _code_lines(pp)
            for j in range(len(lp) - RUN + 1):
                key = tuple(lp[j:j + RUN])
                assert key not in runs, f"{po.name} and {pp.name} share a block starting with: {key[0]}"


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback():
    import paper_2308_04869_b200 as rbg
    import workloads
    with pytest.raises(rbg.RbgError, match="no CUDA device"):
        rbg.Collision(workloads.make(1, np_side=4)["problem"])
