"""Host logic of bench.py on CPU: the max-over-ranks / summed-units aggregation of the replicas-only N > 1 path
(gloo, world_size 2), the algorithmic byte model, and the reference arm's JSON contract."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

RANK_SCRIPT = r"""
import os, sys
sys.path.insert(0, os.environ["MM_ROOT"])
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
dist.init_process_group("gloo", rank=rank, world_size=2)
# rank 0 needs 1.0 s for 100 units, rank 1 needs 2.5 s for 140 units: the job took 2.5 s for 240 units
sec, units = bench.aggregate_over_ranks(1.0 if rank == 0 else 2.5, 100 if rank == 0 else 140)
assert abs(sec - 2.5) < 1e-12 and abs(units - 240.0) < 1e-9, (sec, units)
dist.barrier()
dist.destroy_process_group()
print("rank", rank, "ok")
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_replica_aggregation_gloo_world2():
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), MM_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", RANK_SCRIPT], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    for p in procs:
        out, _ = p.communicate(timeout=240)
        assert p.returncode == 0, out
        assert "ok" in out


def test_algorithmic_bytes_model():
    sys.path.insert(0, ROOT)
    import bench
    from paper_2406_16064_b200 import workloads as wl
    w = wl.cfg4(with_m=False)
    ab = bench.algorithmic_bytes(w, 4)
    assert ab["rhs"] == 89 * w.N * 4 and ab["step"] == (7 * 89 + 102) * w.N * 4 and ab["class"]["y_conv"] == 30 * w.N * 4
    f = wl.cfg5(256, with_m=False)
    ab = bench.algorithmic_bytes(f, 8)
    assert ab["rhs"] == 39 * f.N * 8 and ab["class"]["y_conv"] == 16 * f.N * 8


def test_reference_arm_json_contract():
    """`bench.py --impl reference` times the oracle on a bounded sample and prints the contract's line."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--workload", "cfg5_64"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "cell_updates_per_sec_per_rhs_eval" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["higher_is_better"] is True and line["vs_baseline"] is None


def test_gpus_flag_launches_the_ranks_itself():
    """`bench.py --gpus 2` outside torchrun starts two ranks (torch.distributed.run on 127.0.0.1); in the reference arm
    rank 0 alone works and prints the line with n_gpus = 2, the other rank exits 0."""
    env = dict(os.environ, MM_REF_BUDGET_S="20")
    env.pop("WORLD_SIZE", None); env.pop("RANK", None)
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                          "--workload", "cfg5_64"], capture_output=True, text=True, timeout=900, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(l) for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1 and lines[0]["n_gpus"] == 2 and lines[0]["impl"] == "reference"


def test_world_size_mismatch_is_an_error():
    env = dict(os.environ, WORLD_SIZE="4", RANK="0")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=120, env=env)
    assert out.returncode == 2 and "WORLD_SIZE" in out.stderr


def test_ncu_traffic_lookup_is_keyed_by_version(tmp_path, monkeypatch):
    """roofline.traffic comes from the committed capture table and only for the library version it was captured from."""
    sys.path.insert(0, ROOT)
    import bench
    f = tmp_path / "t.csv"
    f.write_text("# comment\nmm_version,workload,prec,class,kernel,dram_read_bytes,dram_write_bytes,duration_us,capture\n"
                 "v1,cfg4_slab_512x512x16,f32,y_conv,k,100,50,1,c\n")
    monkeypatch.setattr(bench, "TRAFFIC_CSV", str(f))
    assert bench.ncu_traffic("v1", "cfg4_slab_512x512x16", "f32", "y_conv") == 150.0
    assert bench.ncu_traffic("v2", "cfg4_slab_512x512x16", "f32", "y_conv") is None
    assert bench.ncu_traffic("v1", "cfg4_slab_512x512x16", "f64", "y_conv") is None
