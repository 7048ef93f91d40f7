"""Host logic of bench.py for N > 1, on CPU with gloo, world_size 2:
the max-over-ranks reduction of the per-rank time, and that under torchrun only rank 0 of the reference arm
works and prints exactly one JSON line."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
v = bench.max_over_ranks(10.0 + rank, world, "cpu")
assert v == 10.0 + world - 1, v
assert bench.max_over_ranks(3.5, 1, "cpu") == 3.5
dist.barrier()
dist.destroy_process_group()
sys.stdout.write("rank%d-ok-%.1f\n" % (rank, v)); sys.stdout.flush()
"""


def _free_port():
    import socket

    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        return so.getsockname()[1]


def _torchrun(args, timeout=600):
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port)] + args
    env = dict(os.environ, OMP_NUM_THREADS="2")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    assert "rank0-ok-11.0" in r.stdout and "rank1-ok-11.0" in r.stdout, r.stdout


def test_reference_arm_prints_one_line_from_rank0_only():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1", "--config", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0


def test_gpus_flag_alone_starts_the_ranks():
    """`python bench.py --gpus 2` WITHOUT torchrun (the way a user, or a driver, may start it) must become 2 ranks:
    bench.py re-executes itself under torch.distributed.run.  Checked on the reference arm (CPU): rank 0 prints the
    line with n_gpus = 2, the spawned rank 1 exits 0 silently."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    env["OMP_NUM_THREADS"] = "2"
    r = subprocess.run([sys.executable, "bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1",
                        "--config", "1"], cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2


def test_algorithmic_work_charges_masked_and_unmasked_separately():
    """bench.py's roofline numerators from the oracle's split counters: forward charges nothing for
    masked entries (reading 5), backward charges a masked blend dL/dM only."""
    sys.path.insert(0, ROOT)
    import bench

    wc = dict(visible=70, R=1000, fwd_pair_evals=500, fwd_pair_evals_masked=200, fwd_blends=50, fwd_blends_masked=20,
              bwd_pair_evals=480, bwd_pair_evals_masked=190, bwd_blends=48, bwd_blends_masked=19)
    w = bench.algorithmic_work(wc, 100)
    assert w["render_fwd"] == ("alu", 300 * bench.FLOP_PAIR + 30 * bench.FLOP_BLEND_FWD)
    assert w["render_bwd"] == ("alu", 480 * bench.FLOP_PAIR + 29 * bench.FLOP_BLEND_BWD + 19 * bench.FLOP_BLEND_BWD_MASKED)
    assert w["preprocess"] == ("hbm", 70 * 301 + 30 * 109) and w["preprocess_bwd"] == ("hbm", 70 * 513 + 30 * 240)
    assert w["bin_sort"] == ("hbm", 1000 * bench.BYTES_SORT_KEY)


def test_roofline_traffic_is_what_the_tracked_ncu_capture_gives(tmp_path):
    """bench.py's `roofline.traffic` comes from profiles/r03_traffic.json; that file must be exactly what
    ncu_summary.py (beside bench.py) derives from the raw ncu CSV tracked beside it (the number was
    a constant typed into bench.py and could go stale unnoticed), and every call of the hot path must be in it."""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    raw = os.path.join(root, "profiles", "r03_ncu_raw.csv")
    out = tmp_path / "traffic.json"
    subprocess.check_call([sys.executable, os.path.join(root, "ncu_summary.py"), raw, "--config", "3",
                           "--md", str(tmp_path / "table.md"), "--traffic-json", str(out)], cwd=root)
    derived = json.load(open(out))
    tracked = json.load(open(os.path.join(root, "profiles", "r03_traffic.json")))
    assert derived == tracked
    assert set(tracked["3"]) == {"preprocess", "bin_sort", "render_fwd", "render_bwd", "preprocess_bwd"}
    sys.path.insert(0, root)
    import bench

    assert bench.ncu_traffic(3) == tracked["3"]
    # each of the two tables the same script writes has one row per kernel of a step: 22 launches
    table = open(tmp_path / "table.md").read()
    assert sum(1 for ln in table.splitlines() if ln.startswith("| ") and "_kernel" in ln) == 2 * 22
    # north_star's counters for the blend kernels are in it: shared-memory pipe, bank conflicts, red traffic, stalls
    bwd = [ln for ln in table.splitlines() if "render_bwd_kernel" in ln]
    assert len(bwd) == 2 and "short_scoreboard" in bwd[1] and "smem_bank_conflicts" in table and "red_sectors" in table
