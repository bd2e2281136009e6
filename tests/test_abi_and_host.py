"""CPU-side checks of the boundary and of the host logic (no GPU, no compute calls).

* the C-ABI library builds for sm_100a, loads, and exports every function `include/ptycho_b200.h`
  declares;
* calls that need no device behave as documented (defaults, argument errors, workspace sizing);
* `bench.py`'s multi-rank plumbing ("replicas only"): max over ranks and the
  reference arm under a 2-process gloo group.
"""
import ctypes as C
import json
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ptycho_b200.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2202_03144_b200 import binding
    binding.build()
    return binding.lib()


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)          # comments mention names too
    src = re.sub(r"//[^\n]*", "", src)
    return sorted(set(re.findall(r"\b(ptycho_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_paper_step_api():
    names = declared_functions()
    for must in ("ptycho_init", "ptycho_iterate", "ptycho_fetch_object", "ptycho_fetch_probe", "ptycho_fetch_error",
                 "ptycho_workspace_bytes", "ptycho_destroy"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    missing = [n for n in declared_functions() if not hasattr(lib, n)]
    assert not missing, missing


def test_default_params_match_the_readings(lib):
    from paper_2202_03144_b200 import binding
    p = binding.Params()
    lib.ptycho_default_params(C.byref(p))
    assert p.batch_size == 0 and p.probe_start == 0 and p.deterministic == 0 and p.disable_dm == 0
    assert p.delta_blend == pytest.approx(1e-2)              # R5
    assert p.delta_obj == 1.0 and p.delta_probe == 1.0       # R8
    assert p.alpha_obj == 1.0 and p.alpha_probe == 1.0
    assert p.lsq_lambda == pytest.approx(0.1)                # R9
    assert p.pbound == 0.0                                   # R6: exact projection unless asked


def test_workspace_bytes_argument_checks_and_scaling(lib):
    f = lib.ptycho_workspace_bytes
    ok = f(4096, 4096, 256, 1, 10000, 1, 0, None)
    assert ok > 10000 * 256 * 256 * 8                        # holds the DM exit-wave store
    assert f(4096, 4096, 200, 1, 10000, 1, 0, None) == 0     # n not in {64,128,256,512}
    assert f(100, 4096, 256, 1, 10, 1, 0, None) == 0         # object smaller than a frame
    assert f(4096, 4096, 256, 0, 10, 1, 0, None) == 0
    host = f(4096, 4096, 256, 1, 10000, 1, 1, None)          # host intensities are staged in the exit-wave store during init:
    assert host == ok                                        # no extra copy
    from paper_2202_03144_b200 import binding as _b
    nodm = _b.Params()
    lib.ptycho_default_params(C.byref(nodm))
    nodm.disable_dm = 1                                      # without that store they get their own piece
    assert f(4096, 4096, 256, 1, 10000, 1, 1, C.byref(nodm)) - f(4096, 4096, 256, 1, 10000, 1, 0, C.byref(nodm)) == 10000 * 256 * 256 * 2
    stream = f(4096, 4096, 256, 1, 10000, 1, 2, None)        # streaming context: a 64 MB staging piece instead
    assert 0 < stream - ok <= (64 << 20) + (1 << 20)
    from paper_2202_03144_b200 import binding
    p = binding.Params()
    lib.ptycho_default_params(C.byref(p))
    p.disable_dm = 1
    assert f(4096, 4096, 256, 1, 10000, 1, 0, C.byref(p)) < ok - 10000 * 256 * 256 * 8 + (1 << 20)


def test_init_rejects_bad_arguments_before_touching_the_device(lib):
    ctx = C.c_void_p()
    z = np.zeros(8, np.float32)
    st = lib.ptycho_init(C.byref(ctx), None, 64, 64, z.ctypes.data, 1, 64, z.ctypes.data, 1, z.ctypes.data, 0, None, None, 0, None)
    assert st == 1 and not ctx.value                         # PTYCHO_EINVAL, no context
    assert lib.ptycho_iterate(None, 1, 1) == 1
    assert lib.ptycho_launch_count(None) == 0


def test_product_path_has_no_cpu_fallback():
    """The package must not import the oracle, and must raise without a CUDA device."""
    pkg = os.path.join(ROOT, "paper_2202_03144_b200")
    for fn in os.listdir(pkg):
        if fn.endswith(".py"):
            src = open(os.path.join(pkg, fn)).read()
            assert "import oracle" not in src and "from oracle" not in src, fn
    import torch
    if not torch.cuda.is_available():
        from paper_2202_03144_b200 import binding, synth
        s = synth.make_config(0)
        with pytest.raises(Exception):
            binding.Ptycho(s.obj0, s.probe0, s.pos, s.intensities)


# ------------------------------------------------------------------ multi-rank plumbing (gloo, CPU)
WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
r = dist.get_rank()
m = bench.max_over_ranks(10.0 + 5.0 * r, dist.get_world_size())
bench.barrier(dist.get_world_size())
print(json.dumps({{"rank": r, "max": m}}), flush=True)
dist.destroy_process_group()
"""


def run_torchrun(args, port):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port)] + args
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=600)


def test_max_over_ranks_gloo_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    out = run_torchrun([str(script)], 29731)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(l) for l in out.stdout.splitlines() if l.startswith("{")]
    assert sorted(l["rank"] for l in lines) == [0, 1]
    assert all(l["max"] == 15.0 for l in lines)              # the slowest rank's time, on every rank


def test_reference_arm_under_torchrun_prints_one_line_from_rank_0():
    out = run_torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"], 29732)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(l) for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    l = lines[0]
    assert l["impl"] == "reference" and l["cpu_baseline"]["kind"] == "oracle" and l["value"] > 0
    assert l["e2e"]["h2d_bytes_per_step"] == 0 and l["vs_baseline"] is None
