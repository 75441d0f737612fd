"""Host-side logic of bench.py for N > 1 ("replicas only"), on CPU with a world-size-2
gloo group: max-over-ranks timing, whole-job aggregation, and the reference arm under a 2-rank launch
(rank 0 alone runs and prints; the other rank exits 0 without work)."""
import json
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
bench.rank_barrier(world)
ms = bench.rank_max(10.0 + 5.0 * rank, world, "cpu")       # rank 1 is the slow replica
rate = bench.whole_job_rate(1000, 4, world, ms)
sys.stdout.write("RESULT %d %.6f %.6f\n" % (rank, ms, rate)); sys.stdout.flush()   # one write: ranks share the pipe
dist.destroy_process_group()
"""


def _free_port():
    """A port nobody listens on now (a fixed one can still sit in TIME_WAIT from a run a minute ago)."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def _torchrun(args, port=None):
    port = port or _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port)] + args
    env = dict(os.environ, OMP_NUM_THREADS="1")
    return subprocess.run(cmd, cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=300)


def test_max_over_ranks_and_whole_job_rate_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    res = sorted(re.findall(r"RESULT (\d+) ([0-9.]+?\d{6}) ([0-9.]+?\d{6})", r.stdout))
    assert len(res) == 2
    for rank, ms, rate in res:
        assert float(ms) == 15.0                       # every rank sees the slowest replica's time
        assert float(rate) == pytest.approx(2 * 1000 * 4 / 15e-3)


def test_single_rank_helpers_need_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    bench.rank_barrier(1)
    assert bench.rank_max(3.5, 1, "cpu") == 3.5
    assert bench.whole_job_rate(10, 2, 1, 4.0) == pytest.approx(5000.0)


def test_reference_arm_two_ranks_prints_one_line():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload",
                   "sound"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["n_gpus"] == 2 and out["value"] > 0
    assert out["cpu_baseline"]["kind"] == "oracle" and out["e2e"]["h2d_bytes_per_step"] == 0
    assert out["unit"] == "cell updates/s" and out["higher_is_better"] is True


def test_algorithmic_bytes_match_design_table():
    sys.path.insert(0, ROOT)
    import bench
    from paper_1602_02359_b200 import workloads as W
    reals, fused = bench.algorithmic_reals(W.noise_box(shape3=(8, 8, 8)))
    assert 8 * reals["first_sweep"] == 104 and 8 * reals["sweep"] == 136 and 8 * reals["newvel"] == 80
    assert 8 * fused == 464                                   # SURVEY.md 8(d.3), 3-D adiabatic, no FARGO


def test_gpus_2_without_torchrun_launches_two_ranks():
    """`python bench.py --gpus 2` started directly (WORLD_SIZE unset) re-launches itself under torch.distributed.run
    with one process per GPU; the reference arm reaches the same code on CPU: rank 0 prints the one line, n_gpus = 2."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    env["OMP_NUM_THREADS"] = "1"
    r = subprocess.run([sys.executable, "bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                        "--workload", "sound"], cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True,
                       timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1 and json.loads(lines[0])["n_gpus"] == 2


def test_ncu_exports_are_keyed_by_the_kernel_source_hash(tmp_path, monkeypatch):
    """profiling.ncu_table: an export named after the current kernel sources is read as is; one with another hash is
    reported stale; launches of one launcher add up."""
    sys.path.insert(0, ROOT)
    from paper_1602_02359_b200 import profiling as P
    h = P.kernel_source_hash()
    assert len(h) == 10 and h == P.kernel_source_hash()
    head = '"ID","Kernel Name","gpu__time_duration.sum","dram__bytes_read.sum","dram__bytes_write.sum"\n' \
           '"","","ms","Gbyte","Mbyte"\n'
    rows = '"0","void fg::k_sweep_ring<double, (int)1, (int)7>(fg::Dev<double>)","3.5","10","8000"\n' \
           '"1","void fg::k_sweep_ring<double, (int)2, (int)7>(fg::Dev<double>)","3.6","10","8000"\n' \
           '"2","void fg::k_sweep_ring<double, (int)1, (int)7>(fg::Dev<double>)","3.5","10","8000"\n'
    monkeypatch.setattr(P, "PROFILES", str(tmp_path))
    (tmp_path / ("ncu_raw_wl_%s.csv" % h)).write_text(head + rows)
    t, f, stale = P.ncu_table("wl")
    assert stale is False and t["sweep_y"]["launches"] == 2 and t["sweep_z"]["launches"] == 1
    assert t["sweep_y"]["dram_bytes"] == pytest.approx(2 * 18e9) and t["sweep_y"]["ms"] == pytest.approx(7.0)
    (tmp_path / ("ncu_raw_other_0123456789.csv")).write_text(head + rows)
    assert P.ncu_table("other")[2] is True
    assert P.ncu_table("absent") == ({}, None, None)


def test_every_update_kernel_of_the_build_maps_to_a_launcher():
    """profiling.launcher_of joins ncu's kernel names with the launcher names of fargo_profile_report: a kernel of the
    update that maps to nothing would drop out of roofline.traffic silently.  Kernel names come from the tracked SASS
    digest; the exceptions are kernels that run outside an update (field I/O, halo packing, diagnostics, self-test)."""
    import glob
    import re
    sys.path.insert(0, ROOT)
    from paper_1602_02359_b200 import profiling as P
    outside = {"k_copy", "k_gather", "k_scatter", "k_unpad", "k_pad", "k_diagnostics", "k_diag_finish", "k_frame_change",
               "k_selftest_div", "k_halo_pack", "k_halo_unpack", "k_fill"}
    digests = glob.glob(os.path.join(ROOT, "profiles", "sass_digest_*.md"))
    assert digests
    names = set()
    for path in digests:
        for ln in open(path):
            m = re.match(r"\| (k_\w+)(<[^|]*>)? \|", ln)
            if m:
                names.add((m.group(1), (m.group(2) or "").replace("f64", "double").replace("f32", "float")))
    assert len(names) > 40
    unmapped = sorted({n for n, targs in names if n not in outside and P.launcher_of(n + targs) is None})
    assert not unmapped, unmapped
    assert P.launcher_of("void fg::k_sweep_ring<double, (int)1, (int)7>(fg::Dev<double>)") == "sweep_y"
    assert P.launcher_of("void fg::k_mhd_emf<double, (int)2, (int)0>(...)") == "mhd_emf"
    assert P.launcher_of("void fg::k_bc_b<double, (int)1>(...)") == "bc_b" and P.launcher_of("void fg::k_bc<double, (int)1>(...)") == "bc"
