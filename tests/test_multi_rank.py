"""Host-side logic of the N > 1 path of bench.py on CPU: two gloo ranks, each takes its own particle slice
(weak scaling: P per rank fixed, no collective on the data path), the step time is the max over ranks and
the job-wide value is (units of all ranks) / that time.  No GPU needed."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, importlib.util
    import numpy as np, torch, torch.distributed as dist
    sys.path.insert(0, %r)
    import synthetic as syn
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(%r, "bench.py"))
    bench = importlib.util.module_from_spec(spec); spec.loader.exec_module(bench)
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    cfg = syn.CONFIGS[1]
    P = 96
    mine = bench.rank_particles(cfg, P, rank, world)
    assert mine.shape == (P, 6)
    gathered = [torch.zeros(P, 6, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(gathered, torch.as_tensor(mine))
    everything = torch.cat(gathered).numpy()
    # the ranks' slices tile the job's particle set exactly: disjoint, in order, nothing shared
    np.testing.assert_array_equal(everything, syn.draw_particles(cfg, P * world))
    assert len({tuple(r) for r in everything}) == P * world
    # timing: max over ranks; value: units of ALL ranks over that time
    ms = torch.tensor([10.0 + 5.0 * rank], dtype=torch.float64)
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    assert float(ms) == 10.0 + 5.0 * (world - 1)
    n_bins = 1000
    value = float(P) * n_bins * world / (float(ms) * 1e-3)
    assert abs(value - 96 * 1000 * world / ((10.0 + 5.0 * (world - 1)) * 1e-3)) < 1e-6
    dist.barrier()
    dist.destroy_process_group()
    print("rank", rank, "ok")
""") % (ROOT, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_gloo_ranks_shard_particles_without_a_collective_on_the_data_path(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=300)[0] for p in procs]
    for rank, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, out
        assert "rank %d ok" % rank in out


def test_reference_arm_runs_only_on_rank_zero():
    """bench.py --impl reference under torchrun: ranks other than 0 exit 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--config", "tiny"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
