"""CPU-side checks of the boundary and the host logic (no GPU, no compute calls):
 * libaton.so builds (nvcc cross-compiles for sm_100a), loads, and exports every entry point that
   include/aton.h declares; the ctypes structs mirror the header's field order;
 * argument validation that is decided before any CUDA call answers with the documented codes;
 * without a CUDA device aton_init fails loudly (ATON_ECUDA): there is no CPU fallback;
 * the product package never imports oracle/;
 * bench.py's whole-job aggregation (max over ranks of the time, sum of units) under a
   world_size-2 gloo group, which is all the multi-GPU path consists of ("replicas only").
"""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "aton.h")


@pytest.fixture(scope="module")
def lib():
    from paper_1004_2503_b200 import aton, build
    build.build()
    return aton.load_library()


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(aton_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    from paper_1004_2503_b200 import aton
    names = _declared_functions()
    assert {"aton_init", "aton_set_fields", "aton_set_sources", "aton_step", "aton_get_fields",
            "aton_reduce", "aton_courant_dt", "aton_free", "aton_last_error"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"libaton.so does not export {n}"
    assert sorted(aton.EXPORTS) == names
    # the dynamic symbol table holds them as plain C names (no mangling)
    out = subprocess.check_output(["nm", "-D", "--defined-only", aton.LIB_PATH], text=True)
    exported = set(re.findall(r"\bT (aton_[a-z0-9_]+)$", out, flags=re.M))
    assert set(names) <= exported


def test_library_is_sm100a_code(lib):
    from paper_1004_2503_b200 import aton
    out = subprocess.check_output(["/usr/local/cuda/bin/cuobjdump", "-lelf", aton.LIB_PATH], text=True)
    assert "sm_100a" in out


def test_ctypes_structs_mirror_the_header():
    from paper_1004_2503_b200 import aton
    src = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)

    def fields(struct_name):
        body = re.search(r"typedef struct \{([^}]*)\}\s*" + struct_name, src, flags=re.S).group(1)
        names = []
        for decl in body.split(";"):
            decl = decl.strip()
            if not decl:
                continue
            first, *rest = [t.strip() for t in decl.split(",")]
            names.append(first.split()[-1])
            names.extend(rest)
        return names

    assert fields("aton_params_t") == [k for k, _ in aton.Params._fields_]
    assert fields("aton_diag_t") == [k for k, _ in aton.Diag._fields_]
    assert fields("aton_grid_t") == [k for k, _ in aton.Grid._fields_]
    assert fields("aton_box_t") == [k for k, _ in aton.Box._fields_]


def test_argument_validation_without_a_device(lib):
    from paper_1004_2503_b200 import aton, workloads as wl
    h = C.c_void_p()
    p = aton.make_params(wl.default_params())
    box = aton.Box(1e21)
    # bad grid: decided before any CUDA call
    for g in (aton.Grid(10, 8, 8), aton.Grid(0, 8, 8), aton.Grid(8, 0, 8), aton.Grid(2048, 2048, 2048)):
        assert lib.aton_init(C.byref(h), C.byref(g), C.byref(box), C.byref(p), None) == aton.EINVAL
        assert not h.value and lib.aton_last_error(None)
    assert lib.aton_init(C.byref(h), C.byref(aton.Grid(8, 8, 8)), C.byref(aton.Box(0.0)), C.byref(p), None) == aton.EINVAL
    bad = aton.make_params(dict(wl.default_params(), sigma_n=0.0))
    assert lib.aton_init(C.byref(h), C.byref(aton.Grid(8, 8, 8)), C.byref(box), C.byref(bad), None) == aton.EINVAL
    assert lib.aton_init(None, None, None, None, None) == aton.EINVAL
    # NULL contexts never crash
    assert lib.aton_step(None, 1.0, 1) == aton.EINVAL
    assert lib.aton_reduce(None, None) == aton.EINVAL
    assert lib.aton_courant_dt(None, 0.8) < 0
    assert lib.aton_launch_count(None) == 0
    lib.aton_free(None)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device behaviour")
def test_no_cpu_fallback(lib):
    from paper_1004_2503_b200 import aton, workloads as wl
    with pytest.raises(aton.AtonError) as e:
        aton.Aton(8, 8, 8, 1e21, wl.default_params())
    assert e.value.code == aton.ECUDA and "no CPU fallback" in str(e.value)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1004_2503_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "aton_oracle" not in text, f
    o = open(os.path.join(ROOT, "oracle", "aton_oracle.py")).read() + open(os.path.join(ROOT, "oracle", "aton_oracle.c")).read()
    assert "import paper_1004_2503_b200" not in o and "from paper_1004_2503_b200" not in o and "csrc/" not in o.replace(
        "paper_1004_2503_b200/csrc/ and nothing", "")


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=2)
# rank 0 took 100 ms for 1000 units, rank 1 took 250 ms for 3000 units, 5 steps
v, ms = bench.aggregate(100.0 if rank == 0 else 250.0, 1000.0 if rank == 0 else 3000.0, 5, 2)
assert abs(v - 4000.0 / 0.250) < 1e-6 and abs(ms - 50.0) < 1e-9, (v, ms)
assert bench.max_over_ranks(float(rank), 2) == 1.0 and bench.sum_over_ranks(1.5, 2) == 3.0
dist.destroy_process_group()
print("ok", rank)
"""


def test_bench_aggregation_world_size_2_gloo():
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    code = _WORKER.format(root=ROOT, port=port)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1")
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for r, p in enumerate(procs):
        out, _ = p.communicate(timeout=180)
        assert p.returncode == 0 and f"ok {r}" in out, out


def test_bench_reference_arm_runs_on_cpu():
    """`bench.py --impl reference` times the oracle on a bounded sample and prints one JSON line."""
    import json
    out = subprocess.check_output([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                                   "--steps", "2", "--warmup", "3", "--cpu-sample-n", "24",
                                   "--cpu-sample-steps", "4"], text=True, timeout=600)
    line = json.loads(out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["unit"] == "cell-updates/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["higher_is_better"] is True
