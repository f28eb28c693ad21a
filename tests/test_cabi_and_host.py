"""CPU-side checks (-m "not gpu"): libng.so builds/loads and exports every symbol include/ng.h declares; struct
layouts of the binding match the header; the bench's rank-aggregation logic works at world size 2 (gloo)."""
import ctypes as C
import os
import re
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "ng.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ng_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2007_14236_b200 import binding
    L = binding.load_library()
    names = _declared()
    assert len(names) >= 20 and "ng_simulate" in names and "ng_get_state" in names
    for n in names:
        assert hasattr(L, n), n
    assert sorted(binding.EXPORTS) == names


def test_struct_layouts_match_header():
    """Compile a tiny C program against include/ng.h and compare sizeof/offsetof with the ctypes structures."""
    from paper_2007_14236_b200 import binding as B
    prog = textwrap.dedent(r'''
        #include <stdio.h>
        #include <stddef.h>
        #include "ng.h"
        int main(void) {
            printf("%zu %zu %zu %zu %zu\n", sizeof(ng_config), sizeof(ng_lif_params), sizeof(ng_dist), sizeof(ng_stats), sizeof(ng_allocator));
            printf("%zu %zu %zu %zu\n", offsetof(ng_config, seed), offsetof(ng_config, device), offsetof(ng_stats, build_ms), offsetof(ng_stats, delivery_kernel));
            printf("%d %d %d %d %d %d\n", NG_OK, NG_ERR_INVALID_ARG, NG_ERR_STATE, NG_ERR_OOM, NG_ERR_CUDA, NG_ERR_OVERFLOW);
            printf("%d %d %d %d %d %d\n", NG_FIELD_V, NG_FIELD_I_SYN, NG_FIELD_REFR, NG_FIELD_RING, NG_FIELD_STEP, NG_FIELD_LAST_INPUT);
            printf("%d %d %d %d %d %d %d %d %d %d %d\n", NG_OPT_STEP_MODE, NG_OPT_STEPS_PER_GRAPH, NG_OPT_DELIVERY_KERNEL, NG_OPT_DELIVER_BLOCKS, NG_OPT_PROFILE, NG_OPT_ASYNC, NG_OPT_SORT_SEGMENTS, NG_OPT_PREFETCH, NG_OPT_TRACE, NG_OPT_PERSISTENT_THREADS, NG_OPT_QUEUE_CAPACITY);
            return 0;
        }''')
    import tempfile
    with tempfile.TemporaryDirectory() as td:
        c = os.path.join(td, "t.c"); exe = os.path.join(td, "t")
        open(c, "w").write(prog)
        subprocess.check_call(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), c, "-o", exe])   # plain C: the header is C
        out = subprocess.check_output([exe]).decode().split("\n")
    sizes = list(map(int, out[0].split()))
    assert sizes == [C.sizeof(B.NgConfig), C.sizeof(B.NgLifParams), C.sizeof(B.NgDist), C.sizeof(B.NgStats), C.sizeof(B.NgAllocator)]
    offs = list(map(int, out[1].split()))
    assert offs == [B.NgConfig.seed.offset, B.NgConfig.device.offset, B.NgStats.build_ms.offset, B.NgStats.delivery_kernel.offset]
    assert list(map(int, out[2].split())) == [B.NG_OK, B.NG_ERR_INVALID_ARG, B.NG_ERR_STATE, B.NG_ERR_OOM, B.NG_ERR_CUDA, B.NG_ERR_OVERFLOW]
    assert list(map(int, out[3].split())) == [B.FIELD_V, B.FIELD_I_SYN, B.FIELD_REFR, B.FIELD_RING, B.FIELD_STEP, B.FIELD_LAST_INPUT]
    assert list(map(int, out[4].split())) == [B.OPT_STEP_MODE, B.OPT_STEPS_PER_GRAPH, B.OPT_DELIVERY_KERNEL, B.OPT_DELIVER_BLOCKS,
                                              B.OPT_PROFILE, B.OPT_ASYNC, B.OPT_SORT_SEGMENTS, B.OPT_PREFETCH, B.OPT_TRACE, B.OPT_PERSISTENT_THREADS,
                                              B.OPT_QUEUE_CAPACITY]


def test_argument_validation_without_a_gpu():
    """Entry points that need no device reject bad arguments with the documented codes (no compute call)."""
    from paper_2007_14236_b200 import binding as B
    L = B.load_library()
    h = C.c_void_p()
    assert L.ng_create(None, None, None, C.byref(h)) == B.NG_ERR_INVALID_ARG
    bad = B.NgConfig(0.0, 64, 0, 1, 0, 0, 0)
    assert L.ng_create(C.byref(bad), None, None, C.byref(h)) == B.NG_ERR_INVALID_ARG
    bad = B.NgConfig(0.1, 300, 0, 1, 0, 0, 0)
    assert L.ng_create(C.byref(bad), None, None, C.byref(h)) == B.NG_ERR_INVALID_ARG
    assert L.ng_create(C.byref(bad), None, None, None) == B.NG_ERR_INVALID_ARG
    assert L.ng_destroy(None) == B.NG_OK
    assert L.ng_last_error(None) == b"null handle"
    out = C.c_double()
    assert L.ng_probe(0, 7, 1 << 20, C.byref(out)) == B.NG_ERR_INVALID_ARG


def test_product_does_not_import_the_oracle():
    """The product path must not route through oracle/ (only tests, smoke and bench's cpu arms may)."""
    pkg = os.path.join(ROOT, "paper_2007_14236_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "oracle.cpp" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "oracle.cpp")).read()
    assert "paper_2007_14236_b200 import" not in otxt and "ng_device" not in otxt and '#include "ng' not in otxt


def test_sim_refuses_to_run_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    from paper_2007_14236_b200 import binding as B
    with pytest.raises(RuntimeError):
        B.Sim()


_GLOO_WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import torch, torch.distributed as dist
import bench
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
dev = torch.device("cpu")
# rank r "measured" (r+1)*10 ms and delivered (r+1)*1000 events: whole-job time is the max, work is the sum
ms = bench.max_over_ranks(10.0 * (rank + 1), world, dev)
ev = bench.sum_over_ranks(1000.0 * (rank + 1), world, dev)
assert ms == 10.0 * world, ms
assert ev == 1000.0 * world * (world + 1) / 2, ev
wl = bench.make_workload("cfg0", seed_offset=rank)      # replicas use independent seeds
assert wl.seed == 1 + rank
dist.barrier()
dist.destroy_process_group()
sys.stdout.write("ok %d\n" % rank); sys.stdout.flush()   # one write per rank: the two ranks share a pipe
'''


def test_replica_aggregation_world_size_2_gloo(tmp_path):
    """N > 1 path of bench.py (replicas only): max-over-ranks time, sum-over-ranks work, per-rank seeds."""
    script = tmp_path / "w.py"
    script.write_text(_GLOO_WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", "29613", str(script), ROOT]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=240)
    assert out.returncode == 0, out.stderr[-2000:]
    assert "ok 0" in out.stdout and "ok 1" in out.stdout


def test_bench_spawns_its_own_ranks_and_quotes_only_matching_captures(tmp_path, monkeypatch):
    """`python bench.py --gpus N` outside torchrun re-launches itself as N ranks on 127.0.0.1; roofline.traffic is quoted
    from the committed ncu capture only while the kernel sources hash to what the capture was taken on."""
    sys.path.insert(0, ROOT)
    import bench
    cmd = bench.spawn_command(["--gpus", "4", "--steps", "2"], 4, port=29777)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29777"
    assert cmd[-4:] == ["--gpus", "4", "--steps", "2"] and cmd[-5].endswith("bench.py")
    h = bench.csrc_hash()
    f = tmp_path / "t.csv"
    f.write_text(f"# workload,kernel,dram_bytes_per_launch,time_steps_per_launch,csrc_sha256_16,capture\n"
                 f"cfg2,persistent_pipe_kernel,9.0e8,1000,{h},profiles/x.csv\n"
                 f"cfg4,persistent_pipe_kernel,3.6e10,1000,0123456789abcdef,profiles/y.csv\n")
    monkeypatch.setattr(bench, "TRAFFIC_FILE", str(f))
    t, note = bench.ncu_traffic("cfg2", "persistent_pipe_kernel")
    assert t["value"] == 9.0e8 and t["from"] == "profiles/x.csv" and note is None
    t, note = bench.ncu_traffic("cfg4", "persistent_pipe_kernel")
    assert t is None and "0123456789abcdef" in note
    t, note = bench.ncu_traffic("cfg0", "persistent_pipe_kernel")
    assert t is None and note
