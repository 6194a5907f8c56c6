"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/wl_refine.h
declares; host-only pure functions agree with the oracle's independent restatement.  No compute calls (no GPU here)."""
import os
import re

import pytest


def test_library_exports_every_declared_symbol(repo_root):
    import paper_2607_02603_b200 as wl
    from paper_2607_02603_b200.build import build
    build()
    header = open(os.path.join(repo_root, "include", "wl_refine.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(wl_[a-z_0-9]+)\s*\(", header))
    assert declared, "no prototypes found"
    L = wl.lib()
    for name in declared:
        assert hasattr(L, name), f"{name} declared in wl_refine.h but not exported"
    assert declared == set(wl.EXPORTS)


def test_host_weight_function_matches_oracle_restatement():
    import oracle
    import paper_2607_02603_b200 as wl
    for s, st, r, c in [(0, 0, 1, 0), (5, 1, 7, 123456), (2 ** 64 - 1, 9, 3, 2 ** 32 + 5), (42, 1 << 40, 1000, 7)]:
        k = wl.wl_round_key(s, st, r)
        assert k == oracle.round_key(s, st, r)
        assert wl.wl_weight(k, c) == oracle.weight(k, c)


def test_workspace_size_is_monotone_and_rejects_bad_sizes():
    import paper_2607_02603_b200 as wl
    assert wl.wl_refine_workspace_bytes(-1, 0) == 0
    assert wl.wl_refine_workspace_bytes(1 << 40, 0) == 0
    a = wl.wl_refine_workspace_bytes(1000, 5000)
    b = wl.wl_refine_workspace_bytes(2000, 5000)
    c = wl.wl_refine_workspace_bytes(2000, 50000)
    assert 0 < a <= b <= c


def test_no_cpu_fallback_without_cuda():
    import torch
    import paper_2607_02603_b200 as wl
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    import graphgen as gg
    g = gg.erdos_renyi(50, 100, seed=1)
    with pytest.raises(RuntimeError):
        wl.wl_refine(g.n, g.row_ptr, g.col)
    with pytest.raises(RuntimeError):
        wl.wl_refine_host(g.n, g.row_ptr, g.col)


def test_strerror():
    import paper_2607_02603_b200 as wl
    assert wl.wl_strerror(0) == "ok"
    assert "workspace" in wl.wl_strerror(wl.WL_ENOMEM)


def test_deep_and_batched_workspace_sizes():
    import paper_2607_02603_b200 as wl
    base = wl.wl_refine_workspace_bytes(1000, 5000)
    deep = wl.wl_refine_deep_workspace_bytes(1000, 5000)
    # the deep-round regime adds the in-neighbour lists (8(n+1) + 4m) and its work lists
    assert deep >= base + 8 * 1001 + 4 * 5000
    assert wl.wl_refine_deep_workspace_bytes(-1, 0) == 0
    assert wl.wl_refine_deep_workspace_bytes(2000, 5000) >= deep
    # pinned scratch of the batched path: two offset arrays + one weighted entry array
    hb = wl.wl_refine_batched_host_bytes(1000, 5000)
    assert hb >= 2 * 8 * 1001 + 8 * 5000 and wl.wl_refine_batched_host_bytes(-1, 0) == 0


def test_ctypes_structs_mirror_the_header_layout(repo_root, tmp_path):
    """The binding's ctypes structures must have the size and the field offsets gcc gives the structs of include/wl_refine.h
    (a field added on one side only would shift every later field silently)."""
    import ctypes
    import shutil
    import subprocess
    from paper_2607_02603_b200 import binding as B
    if shutil.which("gcc") is None:
        pytest.skip("no gcc")
    structs = {"wl_csr": B.wl_csr, "wl_options": B.wl_options, "wl_stats": B.wl_stats, "wl_edge_batch": B.wl_edge_batch}
    lines = ["#include <stdio.h>", "#include <stddef.h>", '#include "wl_refine.h"', "int main(void) {"]
    for name, cls in structs.items():
        lines.append(f'  printf("{name} %zu\\n", sizeof({name}));')
        for field, _ in cls._fields_:
            lines.append(f'  printf("{name}.{field} %zu\\n", offsetof({name}, {field}));')
    lines += ["  return 0;", "}"]
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", os.path.join(repo_root, "include"), "-o", str(exe), str(src)], check=True)
    got = dict(line.split() for line in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.splitlines())
    header = re.sub(r"/\*.*?\*/", "", open(os.path.join(repo_root, "include", "wl_refine.h")).read(), flags=re.S)
    for name, cls in structs.items():
        assert int(got[name]) == ctypes.sizeof(cls), name
        for field, _ in cls._fields_:
            assert int(got[f"{name}.{field}"]) == getattr(cls, field).offset, f"{name}.{field}"
        body = re.search(r"typedef struct %s \{(.*?)\} %s;" % (name, name), header, flags=re.S).group(1)
        assert len([d for d in body.split(";") if d.strip()]) == len(cls._fields_), f"{name}: field count differs from the header"
