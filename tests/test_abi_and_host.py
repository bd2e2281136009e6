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
sys.stdout.write(json.dumps({{"rank": r, "max": m}}) + "\n"); sys.stdout.flush()       # one write: the ranks share the pipe
dist.destroy_process_group()
"""


def json_objects(text):
    """The flat JSON objects in a stream that several ranks wrote to (their lines can run into each other)."""
    import re
    return [json.loads(m) for m in re.findall(r"\{[^{}]*\}", text)]


def run_torchrun(args, port):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port)] + args
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=600)


def test_max_over_ranks_gloo_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    out = run_torchrun([str(script)], 29731)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = json_objects(out.stdout)
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


# ------------------------------------------------------------------ one scan over several GPUs: plan and exchange
def _scan_positions(rng, J, n, H, W):
    return np.stack([rng.integers(0, H - n + 1, J), rng.integers(0, W - n + 1, J)], 1).astype(np.int32)


@pytest.mark.parametrize("world,J,n,H,W,seed", [(1, 40, 16, 90, 70, 0), (2, 57, 16, 120, 80, 1), (3, 200, 32, 300, 260, 2),
                                                (4, 31, 64, 200, 200, 3), (8, 8, 16, 40, 40, 4)])
def test_shard_plan_against_brute_force(world, J, n, H, W, seed):
    """The plan is integer work: every property is checked against its definition, pixel row by pixel row."""
    from paper_2202_03144_b200.sharded import shard_plan
    rng = np.random.default_rng(seed)
    pos = _scan_positions(rng, J, n, H, W)
    pl = shard_plan(pos, n, H, W, world)
    allf = np.concatenate(pl.frames)
    assert sorted(allf.tolist()) == list(range(J))                                   # a partition of the frames
    assert max(len(f) for f in pl.frames) - min(len(f) for f in pl.frames) <= 1      # balanced
    cover = np.zeros((world, H), bool)                                               # rows each rank's frames touch
    for r in range(world):
        for j in pl.frames[r]:
            cover[r, pos[j, 0]:pos[j, 0] + n] = True
        lo, hi = pl.rows[r]
        assert cover[r, lo] and cover[r, hi - 1] and not cover[r, :lo].any() and not cover[r, hi:].any()
        # foreign frames: exactly the other ranks' frames with a row inside [lo, hi)
        want = sorted(j for q in range(world) if q != r for j in pl.frames[q] if pos[j, 0] < hi and pos[j, 0] + n > lo)
        assert pl.foreign[r].tolist() == want
        # every pixel row of an own frame gets d_O from every frame of the scan that covers it
        mine_or_foreign = set(pl.frames[r].tolist()) | set(want)
        for y in range(lo, hi):
            covering = {j for j in range(J) if pos[j, 0] <= y < pos[j, 0] + n}
            assert covering <= mine_or_foreign
    for r in range(world):                                                           # exchange lists: symmetric, exact row ranges
        for q, a, b in pl.exchange[r]:
            assert (r, a, b) in pl.exchange[q]
            assert (a, b) == (max(pl.rows[r][0], pl.rows[q][0]), min(pl.rows[r][1], pl.rows[q][1])) and a < b
        for q in range(world):
            if q != r and not any(e[0] == q for e in pl.exchange[r]):
                assert min(pl.rows[r][1], pl.rows[q][1]) <= max(pl.rows[r][0], pl.rows[q][0])
    own = np.zeros(H, int)                                                           # owned rows: disjoint, inside the rank's band, together
    for r in range(world):                                                           # the union of all bands
        lo, hi = pl.owned[r]
        assert pl.rows[r][0] <= lo <= hi <= pl.rows[r][1]
        own[lo:hi] += 1
    band = np.zeros(H, bool)
    for lo, hi in pl.rows:
        band[lo:hi] = True
    assert (own[band] == 1).all() and (own[~band] == 0).all()


SHARD_WORKER = r"""
import sys, json, numpy as np, torch
sys.path.insert(0, {root!r})
import torch.distributed as dist
from paper_2202_03144_b200.sharded import shard_plan, HaloExchange, DistComm, stitch_rows
dist.init_process_group("gloo")
comm = DistComm()
r, world = comm.rank, comm.world
rng = np.random.default_rng(5)
n, H, W, J = 16, 96, 40, 61
pos = np.stack([rng.integers(0, H - n + 1, J), rng.integers(0, W - n + 1, J)], 1).astype(np.int32)
pl = shard_plan(pos, n, H, W, world)
def partial(rank):                       # a rank's part of an overlap sum: integers inside its band, zero outside (exact in fp32)
    g = np.random.default_rng(100 + rank)
    c = np.zeros((H, W, 2), np.float32)
    lo, hi = pl.rows[rank]
    c[lo:hi] = g.integers(-1000, 1000, (hi - lo, W, 2))
    return c
c = torch.from_numpy(partial(r))
HaloExchange(pl, r).run(c, comm)
total = sum(partial(q) for q in range(world))
lo, hi = pl.rows[r]
ok_rows = bool((c[lo:hi].numpy() == total[lo:hi]).all())
probe = torch.full((12,), float(r + 1)); comm.all_reduce(probe)
fill = torch.full((H, W, 2), -7.0)
term = stitch_rows(pl, r, c, fill); comm.all_reduce(term)
band = np.zeros(H, bool)
for a, b in pl.rows: band[a:b] = True
ok_stitch = bool((term.numpy()[band] == total[band]).all() and (term.numpy()[~band] == -7.0).all())
sys.stdout.write(json.dumps({{"rank": r, "rows": ok_rows, "probe": float(probe[0]), "stitch": ok_stitch, "peers": len(pl.exchange[r])}}) + "\n"); sys.stdout.flush()
dist.destroy_process_group()
"""


def test_halo_exchange_gloo_world_size_2(tmp_path):
    """The exchange step of the sharded run (neighbour send / receive of row blocks, all-reduce, stitching) under a real
    2-process group on CPU tensors: afterwards every rank holds the TOTAL of the partial canvases on every row of its band."""
    script = tmp_path / "shard_worker.py"
    script.write_text(SHARD_WORKER.format(root=ROOT))
    out = run_torchrun([str(script)], 29733)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = json_objects(out.stdout)
    assert sorted(l["rank"] for l in lines) == [0, 1]
    assert all(l["rows"] and l["stitch"] and l["probe"] == 3.0 and l["peers"] == 1 for l in lines)


def test_halo_exchange_without_peers_is_a_no_op():
    import torch
    from paper_2202_03144_b200.sharded import shard_plan, HaloExchange
    pos = np.array([[0, 0], [5, 3], [9, 9]], np.int32)
    pl = shard_plan(pos, 16, 40, 40, 1)
    c = torch.arange(40 * 40 * 2, dtype=torch.float32).view(40, 40, 2)
    ref = c.clone()
    h = HaloExchange(pl, 0)
    for _ in range(2):                                       # twice: the staging list is reused
        h.run(c, comm=None)
    assert torch.equal(c, ref) and pl.owned == [(0, 25)] and pl.foreign[0].size == 0
