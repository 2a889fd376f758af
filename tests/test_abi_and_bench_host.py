"""Host-side checks that need no GPU: libepic.so builds, loads and exports every symbol that
include/epic.h declares; bench.py's cost model against the one number the paper prints for it;
the multi-rank reduction bench.py uses, on gloo with world_size 2."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "epic.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"EPIC_API\s+[\w\s\*]+?\b(epic_\w+)\s*\(", text)))


def test_header_declares_the_north_star_trio():
    names = _declared_symbols()
    for n in ("epic_plan_create", "epic_image", "epic_plan_destroy"):
        assert n in names
    assert len(names) >= 10


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1904_11422_b200.build import build
    path = build()  # no-op when libepic.so is newer than its sources
    handle = ctypes.CDLL(path)
    for name in _declared_symbols():
        assert hasattr(handle, name), f"{name} declared in include/epic.h but not exported"
    import paper_1904_11422_b200 as epic
    assert sorted(epic.SYMBOLS) == _declared_symbols()  # the binding covers the whole header
    # pure host entry points can be called without a GPU
    assert epic.lib().epic_status_string(0) == b"EPIC_OK"
    assert b"ARG" in epic.lib().epic_status_string(-1)
    assert epic.lib().epic_plan_destroy(None) == 0
    assert epic.lib().epic_plan_get_n(None) == epic.EPIC_ERR_ARG


def test_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1904_11422_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f"{f} mentions the oracle"


def test_fft_cost_model_matches_the_papers_ratio():
    sys.path.insert(0, ROOT)
    import bench
    from workloads import make_custom
    row = [l for l in open(os.path.join(ROOT, "tests", "golden", "paper_fft_cost_ratio.txt"))
           if not l.startswith("#")][0].split()
    n0, n1, ratio, tol = int(row[0]), int(row[1]), float(row[2]), float(row[3])

    def fft_flops(n):  # pad = 1: no pruning, so only the N^2 log2 N^2 term is left besides S3/S5
        wl = make_custom(grid_n=n, pad=1, n_ant=1, n_pol=1, kernel_k=1, n_chan=1, n_t=1)
        return bench.algorithmic_flops_per_frame(wl) - 2.0 - 4.0 * n * n

    assert abs(fft_flops(n1) / fft_flops(n0) - ratio) <= tol
    assert fft_flops(64) == pytest.approx(5.0 * 64 * 64 * 12)


_WORKER = r"""
import os, sys, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
import bench
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=2)
r = dist.get_rank()
out = bench.max_over_ranks([10.0 + r, 5.0 - r], torch.device("cpu"))
assert out == [11.0, 5.0], out
lo, hi = bench.channel_shard(128, r, 2)
assert (lo, hi) == ((0, 64) if r == 0 else (64, 128))
dist.destroy_process_group()
print("ok", r)
"""


def test_multi_rank_reduction_and_sharding_on_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29571", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script), ROOT], env=dict(env, RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True) for r in range(2)]
    outs = [p.communicate(timeout=120)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o


def test_bench_per_channel_variant_keeps_the_configs_shape():
    import bench
    from workloads import make_config
    base = make_config(3, n_chan=4, n_t=6)
    pc = bench.per_channel_variant(base)
    assert pc.ant_uv.shape == (4, 256, 2) and pc.taps.shape == (4, 256, 3, 3, 2)
    assert (pc.grid_n, pc.pad, pc.n_pol, pc.n_products, pc.n_t, pc.index) == (64, 2, 2, 4, 6, 3)
    # 25 kHz channels from 38 MHz: coordinates relative to the centre grow by 25/38000 per channel
    off = pc.ant_uv.astype(np.float64) - 32.0
    np.testing.assert_allclose(off[3], off[0] * (38e6 + 75e3) / 38e6, rtol=1e-4, atol=1e-4)
    assert bench.algorithmic_flops_per_frame(pc) == bench.algorithmic_flops_per_frame(base)
    assert pc.voltages().shape == (6, 4, 2, 256)


def test_binding_rejects_host_tensors_for_device_pointers():
    """binding._check_tensor: a CPU tensor, a wrong dtype or a short buffer never reaches the C ABI."""
    import pytest
    import torch
    from paper_1904_11422_b200 import binding
    with pytest.raises(ValueError):
        binding._check_tensor(torch.zeros(16, dtype=torch.uint8), "voltages", "uint8", 16, None)
    binding._check_tensor(1234, "voltages", "uint8", 16, None)   # raw addresses are the caller's business, as in C
    binding._check_tensor(None, "voltages", "uint8", 16, None)


def test_header_is_plain_c_and_a_c_program_links_and_fails_loudly_without_a_gpu(tmp_path):
    """include/epic.h is a C ABI: it compiles as C99 with gcc, a C program links against libepic.so with no C++ or
    torch in sight, and without a CUDA device the library reports EPIC_ERR_CUDA (there is no CPU fallback); with a
    device the same program succeeds."""
    import shutil
    import subprocess
    from paper_1904_11422_b200 import binding
    from paper_1904_11422_b200.build import build
    gcc = shutil.which("gcc")
    if gcc is None:
        import pytest
        pytest.skip("no gcc")
    build()
    inc = os.path.join(ROOT, "include")
    subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-fsyntax-only", "-x", "c",
                    os.path.join(inc, "epic.h")], check=True)
    src = tmp_path / "use_epic.c"
    src.write_text('#include "epic.h"\n#include <stdio.h>\n'
                   'int main(void) {\n  epic_plan* p = 0;\n  float uv[2] = {1.0f, 2.0f};\n'
                   '  int st = epic_plan_create(&p, 16, 2, 1, uv, 0, 1);\n'
                   '  printf("%d|%s|%lld\\n", st, epic_status_string(st), epic_noalloc_scratch_bytes());\n'
                   '  epic_plan_destroy(p);\n  return 0;\n}\n')
    exe = tmp_path / "use_epic"
    libdir = os.path.dirname(binding.LIB_PATH)
    subprocess.run([gcc, "-std=c99", "-Wall", "-I", inc, str(src), "-o", str(exe), "-L", libdir, "-l:libepic.so",
                    f"-Wl,-rpath,{libdir}"], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.strip().split("|")
    assert int(out[0]) in (binding.EPIC_OK, binding.EPIC_ERR_CUDA), out
    assert out[1].startswith("EPIC_OK") or out[1].startswith("EPIC_ERR_CUDA"), out
    assert int(out[2]) == 80 << 20
