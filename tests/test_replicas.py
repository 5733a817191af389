"""The N > 1 path of bench.py on CPU: two gloo ranks run the replica plumbing (barrier, MAX over
ranks, whole-job throughput, view sharding).  No kernel runs here: the data path has no collective."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, sys
    sys.path.insert(0, %r)
    from paper_2606_18588_b200 import replicas
    world, rank = replicas.init("gloo")
    assert world == 2
    replicas.barrier(cuda=False)
    ms = 2.0 + 3.0 * rank                       # rank 1 is slower
    thr, ms_max = replicas.whole_job_throughput(1000.0 * (rank + 1), ms, cuda=False)
    out = dict(rank=rank, ms_max=ms_max, thr=thr, views=replicas.shard_views(5, world, rank),
               seed=replicas.replica_view_seed(2, rank), mx=replicas.max_over_ranks(float(rank), False))
    replicas.barrier(cuda=False)
    replicas.finish()
    print("RESULT " + json.dumps(out))
""") % ROOT


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_gloo_ranks_agree_on_max_time_and_whole_job_throughput(tmp_path):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(r), LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        so, se = p.communicate(timeout=180)
        assert p.returncode == 0, se
        outs.append(json.loads([l for l in so.splitlines() if l.startswith("RESULT ")][0][7:]))
    outs.sort(key=lambda o: o["rank"])
    for o in outs:
        assert o["ms_max"] == 5.0                         # MAX over ranks, not this rank's time
        assert abs(o["thr"] - 3000.0 / 5e-3) < 1e-6       # all ranks' units / max time
        assert o["mx"] == 1.0
    assert outs[0]["views"] == [0, 2, 4] and outs[1]["views"] == [1, 3]
    assert outs[0]["seed"] != outs[1]["seed"]


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    from paper_2606_18588_b200 import replicas
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK"):
        os.environ.pop(k, None)
    assert replicas.world_info() == (1, 0, 0)
    assert replicas.max_over_ranks(3.5, cuda=False) == 3.5
    thr, ms = replicas.whole_job_throughput(10.0, 2.0, cuda=False)
    assert ms == 2.0 and thr == 5000.0


def test_bench_reference_arm_prints_only_on_rank_0():
    """`bench.py --impl reference` under torchrun: rank != 0 exits 0 without work or output."""
    env = dict(os.environ, WORLD_SIZE="2", RANK="1", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
