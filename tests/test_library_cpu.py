"""CPU-side checks of the C-ABI library and the host logic: no GPU, no compute calls.

 * libchfsi.so builds/loads and exports every function include/chfsi.h declares;
 * argument errors are reported through the ABI's status codes (they are checked before any device work);
 * without a CUDA device the product path fails LOUDLY (there is no CPU fallback);
 * the band-parallel sharding helpers, single-process and under a 2-rank gloo group.
"""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    with open(os.path.join(ROOT, "include", "chfsi.h")) as f:
        text = f.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(chfsi_[a-zA-Z0-9_]+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    from paper_2203_07820_b200 import EXPORTED_SYMBOLS, load_library
    lib = load_library()
    names = declared_functions()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/chfsi.h but not exported by libchfsi.so"
    assert sorted(EXPORTED_SYMBOLS) == names


def test_library_links_only_cuda_runtime_not_torch_or_python():
    from paper_2203_07820_b200.binding import LIB_PATH
    out = subprocess.run(["ldd", LIB_PATH], capture_output=True, text=True).stdout
    needed = [line.split()[0] for line in out.splitlines() if line.strip()]
    assert any(n.startswith("libcudart") for n in needed)
    assert not any("torch" in n or "libpython" in n or "c10" in n for n in needed), needed


def _has_gpu():
    import torch
    return torch.cuda.is_available()


def test_argument_errors_come_back_as_status_codes():
    from paper_2203_07820_b200 import load_library
    from paper_2203_07820_b200.binding import _Mesh, _Potential
    lib = load_library()
    h = C.c_void_p()
    assert lib.chfsi_create(None, None, None, None, 64, 0, None) == -1
    cd = np.zeros((1, 8), dtype=np.int32)
    cv = np.zeros((1, 8, 3))
    vq = np.zeros((1, 27))
    mesh = _Mesh(1, 1, 8, cd.ctypes.data, cv.ctypes.data)
    pot = _Potential(vq.ctypes.data)
    assert lib.chfsi_create(C.byref(h), C.byref(mesh), C.byref(pot), None, 16, 0, None) == -5   # precision
    assert b"precision" in lib.chfsi_last_error(None)
    mesh9 = _Mesh(9, 1, 8, cd.ctypes.data, cv.ctypes.data)
    assert lib.chfsi_create(C.byref(h), C.byref(mesh9), C.byref(pot), None, 64, 0, None) == -5  # p > 8
    assert lib.chfsi_create(C.byref(h), C.byref(mesh), C.byref(pot), None, 64, 7, None) == -1   # assembly
    assert lib.chfsi_create(C.byref(h), C.byref(mesh), None, None, 64, 0, None) == -1           # NULL potential
    assert h.value is None
    # NULL handles
    assert lib.chfsi_destroy(None) == -1
    assert lib.chfsi_apply_H(None, None, 0, None, 0, 0, None, None) == -1
    assert lib.chfsi_chebyshev_filter(None, None, 0, 0, 1, 0.0, 1.0, 0.0, None, None) == -1
    assert lib.chfsi_launch_count(None) == -1


@pytest.mark.skipif(_has_gpu(), reason="checks the no-device behaviour")
def test_no_cpu_fallback_without_a_device():
    from paper_2203_07820_b200 import ChfsiError, Operator, load_library
    from paper_2203_07820_b200.binding import _Mesh, _Potential
    from workloads.generate import make_workload
    wl = make_workload(None, n=2, p=1, L=2.0, atoms_per_side=1, n_gaussians=0, nonlocal_=False, smooth_field=0.0,
                       seed_base=1)
    with pytest.raises(ChfsiError):
        Operator.from_workload(wl)
    lib = load_library()
    h = C.c_void_p()
    cd = np.ascontiguousarray(wl.cell_dofs)
    mesh = _Mesh(1, wl.n_cells, wl.n_dofs, cd.ctypes.data, wl.cell_vertices.ctypes.data)
    pot = _Potential(wl.veff_q.ctypes.data)
    assert lib.chfsi_create(C.byref(h), C.byref(mesh), C.byref(pot), None, 64, 0, None) == -4    # CHFSI_ERR_CUDA
    assert b"no CPU fallback" in lib.chfsi_last_error(None)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2203_07820_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cpp", ".h")):
                with open(os.path.join(dirpath, fn)) as f:
                    src = f.read()
                assert "oracle" not in src.replace("no oracle", ""), f"{fn} mentions the oracle"


def test_column_shard_partitions_the_columns():
    from paper_2203_07820_b200.sharding import column_shard
    for n, w, mult in [(1024, 4, 8), (4000, 8, 8), (10, 3, 1), (5, 8, 1), (0, 2, 1), (4096, 2, 512)]:
        pieces = [column_shard(n, w, r, mult) for r in range(w)]
        assert pieces[0][0] == 0 and pieces[-1][1] == n
        for (a0, a1), (b0, b1) in zip(pieces, pieces[1:]):
            assert a1 == b0 and a0 <= a1
        sizes = [j1 - j0 for j0, j1 in pieces]
        assert max(sizes) - min(s for s in sizes) <= mult or n < w * mult
        assert all(j0 % mult == 0 for j0, j1 in pieces if j1 > j0)
    with pytest.raises(ValueError):
        column_shard(8, 2, 2)


_GLOO_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
from paper_2203_07820_b200.sharding import aggregate_max, column_shard
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
r = dist.get_rank()
j0, j1 = column_shard(1000, 2, r, 8)
# each rank reports its own range and a rank-dependent "time"; the max must be the slow rank's on both
t = aggregate_max(10.0 + 5.0 * r, 2)
tot = aggregate_max(float(j1 - j0), 2)
assert t == 15.0, t
assert (j0, j1) == ((0, 504) if r == 0 else (504, 1000)), (j0, j1)
assert tot == 504.0
dist.barrier()
dist.destroy_process_group()
print("ok", r)
"""


def test_band_parallel_helpers_under_gloo_world_size_2(tmp_path):
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    script = tmp_path / "worker.py"
    script.write_text(_GLOO_WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {r}" in o, o
