"""CPU-side checks of the boundary: libqcf.so builds for sm_100a, loads without a GPU, exports every symbol that
include/qcf.h declares, and its host-only entry points behave (no compute calls here)."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_05875_b200 import binding, build
    build.build()
    return binding.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "qcf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"QCF_API\s+[\w\s\*]+?\b(qcf_\w+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    from paper_2606_05875_b200 import binding
    declared = _declared_symbols()
    assert len(declared) >= 15
    assert sorted(binding.EXPORTS) == declared, "binding.EXPORTS must list exactly what qcf.h declares"
    for name in declared:
        assert hasattr(lib, name), name
    # and nothing else leaks out of the shared object
    out = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l and not l.split()[-1].startswith("_"))
    assert exported == declared


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "qcf.h"\nint main(void) { qcf_layout l; qcf_layer_args a; (void)l; (void)a; return 0; }\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src), "-o",
                    str(tmp_path / "t.o")], check=True)


def test_library_is_sm100a_with_expected_kernels():
    """The shipped cubin is sm_100a and its kernels are what DESIGN.md says they are (profiles/r03_sass_census.md holds the
    same census as a table): the contractions issue tcgen05.mma (UTCHMMA) with TMEM loads (LDTM) and TMA tensor loads
    (UTMALDG), the streaming kernels move rows with bulk async copies (UBLKCP), and no legacy mma.sync (HMMA) exists."""
    from paper_2606_05875_b200 import binding
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run(["cuobjdump", "-sass", binding.LIB_PATH], capture_output=True, text=True).stdout
    census = {}
    for part in re.split(r"\n\s*Function : ", sass)[1:]:
        name = part.split("\n", 1)[0].strip()
        census[name] = {op: len(re.findall(r"\b" + op, part)) for op in ("UTCHMMA", "LDTM", "UTMALDG", "UBLKCP", "HMMA")}
    assert len(census) >= 40

    def of(kernel):
        rows = [c for n, c in census.items() if re.search(r"\d+" + kernel + r"(I|E)", n)]
        assert rows, kernel
        return rows

    for kernel in ("attn_tc_kernel", "score_tc_kernel", "gemm_tc_kernel"):
        for c in of(kernel):
            assert c["UTCHMMA"] > 0 and c["LDTM"] > 0 and c["UTMALDG"] > 0, (kernel, c)
    for kernel in ("reposition_tma_kernel", "scatter_tma_kernel", "gather_rows_tma_kernel"):
        for c in of(kernel):
            assert c["UBLKCP"] > 0, (kernel, c)
    assert sum(c["HMMA"] for c in census.values()) == 0, "a legacy mma.sync path crept in"


def test_n_select_floor_rule(lib):
    # DESIGN.md reading (g): floor(rho N + 1e-6) in double; the BASELINE configs' values
    cases = [(128, 0.3, 38), (5120, 0.3, 1536), (10240, 0.3, 3072), (8192, 0.1, 819), (8192, 0.3, 2457),
             (8192, 0.5, 4096), (32768, 0.15, 4915), (10, 0.0, 0), (10, 1.0, 10), (0, 0.5, 0)]
    for n, r, k in cases:
        assert lib.qcf_n_select(n, r) == k
    assert lib.qcf_n_select(-1, 0.5) == -1 and lib.qcf_n_select(5, 1.5) == -1 and lib.qcf_n_select(5, float("nan")) == -1


def test_create_fails_loudly_without_device_or_on_bad_layout(lib):
    from paper_2606_05875_b200 import binding
    import torch
    h = ctypes.c_void_p()
    lay = binding.qcf_layout(8, 3, 128, 1e6, 0.0)                  # Hkv does not divide Hq
    assert lib.qcf_create(ctypes.byref(h), ctypes.byref(lay), 1, 128, 8) == binding.QCF_ERR_UNSUPPORTED
    assert b"divide" in lib.qcf_last_error(None)
    if not torch.cuda.is_available():
        lay = binding.qcf_layout(8, 2, 128, 1e6, 0.0)
        st = lib.qcf_create(ctypes.byref(h), ctypes.byref(lay), 1, 128, 8)
        assert st == binding.QCF_ERR_UNSUPPORTED and not h.value, "no CPU fallback: creation must fail without a GPU"
        with pytest.raises(binding.QcfError):
            binding.Context(8, 2, 128, 1e6, 1, 128, 8)


def test_bench_reference_arm_under_two_gloo_ranks(tmp_path):
    """The N > 1 launch contract on CPU: `torch.distributed.run` with two ranks (no GPU, gloo rendezvous on 127.0.0.1):
    rank 0 alone runs the reference arm and prints ONE JSON line, the other rank exits 0 without work."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29731", os.path.join(root, "bench.py"), "--impl", "reference", "--workload", "c1", "--gpus", "2",
           "--steps", "2", "--warmup", "1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0


def test_max_over_ranks_two_gloo_ranks():
    """bench.py reduces its timings with a MAX over ranks; the same reduction on a 2-rank gloo group."""
    import torch.multiprocessing as mp
    mp.spawn(_gloo_worker, args=(2, 29733), nprocs=2, join=True)


def _gloo_worker(rank, world, port):
    import torch
    import torch.distributed as dist
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    import bench
    t = bench.max_over_ranks([10.0 + rank, 3.0 - rank], dist, "cpu")
    assert t == [11.0, 3.0], t
    dist.barrier()
    dist.destroy_process_group()
