"""N > 1 host logic of bench.py on CPU (gloo, world_size 2): replicas only, max-over-ranks timing,
whole-job aggregate, and the reference arm printing on rank 0 only."""
import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        ms_local = 10.0 + 5.0 * rank              # rank 1 is the slow replica
        dist.barrier()
        ms = bench.max_over_ranks(ms_local, world, "cpu")
        value = bench.whole_job_value(world, dofs_stage=1000, steps=4, seconds=ms * 1e-3)
        Path(out_dir, f"rank{rank}.json").write_text(json.dumps({"ms": ms, "value": value}))
    finally:
        dist.destroy_process_group()


def test_replicas_max_over_ranks_gloo(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    outs = [json.loads((tmp_path / f"rank{r}.json").read_text()) for r in range(2)]
    for o in outs:
        assert o["ms"] == 15.0                                   # the slowest replica's time on every rank
        assert o["value"] == pytest.approx(2 * 1000 * 4 / 15.0e-3)  # whole-job aggregate over both replicas


def test_reference_arm_rank0_only():
    """bench.py --impl reference under a 2-rank launch: rank 0 runs the oracle and prints one JSON
    line, the other rank exits 0 without work (no process group is needed for it)."""
    outs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(_free_port()))
        r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2",
                            "--warmup", "1", "--workload", "C1"], capture_output=True, text=True, env=env, timeout=300)
        assert r.returncode == 0, r.stderr[-2000:]
        outs.append(r.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["config"]["workload"].startswith("C1")


def test_bench_spawns_its_own_ranks_when_not_under_torchrun():
    """`python bench.py --gpus 2` with no torchrun environment re-executes itself under torch.distributed.run with two
    ranks (rendezvous on 127.0.0.1) and the line says n_gpus = 2 (it used to run one replica and say 1).
    Checked here with the reference arm, which needs no GPU; the GPU arm takes the same path."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "1",
                        "--workload", "C1"], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                       # rank 0 alone prints
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["impl"] == "reference"


def test_both_arms_name_the_workload_with_the_same_config_keys():
    """The driver compares the two arms' `config` dicts: both come from bench.workload_config."""
    sys.path.insert(0, str(ROOT))
    import bench
    w = bench.make_workload("C1")
    cfg = bench.workload_config(w)
    assert set(cfg) == {"workload", "n_elem", "n_edge", "n_nodes", "p", "rk_order", "dt", "limiter", "wetdry", "flux", "wind", "tide", "l2"}
    src = (ROOT / "bench.py").read_text()
    assert src.count('"config": workload_config(w)') + src.count('"config": cfg') >= 2


def test_bench_bookkeeping_plain_stages_and_traffic_table():
    """Roofline bookkeeping of bench.py: the number of stages that do not read w^n follows the scheme (1 for SSP(2,2) and
    SSP(3,3), s-1 for SSP(s,2), 3 for SSP(4,3)), and profiles/traffic.csv parses into per-(workload, kernel) records that
    name their ncu capture."""
    import bench
    from workloads import c1
    from workloads.configs import Workload

    def with_rk(order, stages):
        w = c1(nq=4)
        prm = dict(w.params); prm.update(rk_order=order, rk_stages=stages)
        return Workload(w.name, w.mesh, w.bathy, prm, w.ze, w.qx, w.qy, w.dt, w.nsteps)

    assert [bench.plain_stages(with_rk(o, s)) for o, s in ((2, 0), (3, 0), (2, 3), (2, 4), (3, 4))] == [1, 1, 2, 3, 3]
    tr = bench.read_traffic()
    rec = tr[("C3", "stage")]
    assert rec["dram_bytes"] > 1e9 and rec["source"] and rec["fp64_inst_per_elem"] > 100
    assert all(v["source"] for v in tr.values())
    w = bench.make_workload("C1+perturbed")
    assert w.name.endswith("+perturbed") and abs(w.qx).max() > 0
